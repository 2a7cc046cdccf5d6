// sweep.cuh -- the level sweep of the CUDA path: one fused kernel per level update
// (rows a1, a6-a9 of SURVEY.md Sec. 8(a) around the cell-local arithmetic of collide.cuh).
//
// One thread updates one cell (pull scheme, Eq. 31): it reads its Q-1 links from the
// direction-major int32 list (coalesced), gathers Q (2Q) populations from the level's old buffer,
// resolves wall / velocity-bounce-back links from its own old populations, and
//   FLUID / NEUMANN   collides and stores to its own slot of the new buffer (coalesced);
//   COARSE_GHOST      first coalesces its unknown directions from its children's current values
//                     (Eq. 4, 6 P:104-118), collides once (S15), stores, and explodes the result to
//                     its <= 4 children on the finer level (Eq. 5, 7 P:108-122);
//   FINE_GHOST        stores what it gathered, without colliding;
//   DIRICHLET         stores the equilibrium of the imposed state.
// Each thread writes only its own slot (and its own children), so there are no atomics and no
// write hazards; the two-buffer scheme of the paper is kept.
// BRICKS kernels put a second addressing in front of that list path: regular 8x8 tiles of fluid cells ("bricks",
// verified against the list by the host builder) are updated by the first CTAs of the same launch through tile
// arithmetic, without list, type or link handling (brick_update below).
#pragma once
#include "collide.cuh"

namespace lbm {

constexpr int TYPE_MASK = 7;     // low bits of the device type byte = LBM_* cell type
constexpr int TYPE_SIDE_SHIFT = 4;  // boundary cells: side in bits 4-5

// Kernel arguments are plain structs with untyped pointers (the precision is a template parameter of
// the kernel, not of its arguments), so that the host side launches every instantiation the same way.
struct LevelArgs {
  int n;                    // stored cells of this level
  long long ps;             // plane stride of the population arrays and of the list (elements)
  const void* So;           // old buffer  [npop][ps]
  void* Sn;                 // new buffer
  const int* nbr;           // [(Q-1)][ps] pull sources / negative link codes
  const unsigned char* type;
  const int* aux;           // ghost index (coarse ghost) / source cell (boundary cells)
  const int* g_child;       // [ng][4] children on the finer level
  void* fine;               // finer level's CURRENT buffer (coalescence reads, explosion writes)
  long long fps;            // its plane stride
  double tau;
  const double* sigma;      // sponge coefficient per cell (Eq. 11) or null
  int* status;              // sticky FLAG_* word
  // compressed addressing (BRICKS kernels): the first list_ctas CTAs update the n_irr irregular cells irr[] through the
  // list (first, so that the slower one-cell-per-thread work is not the tail of the launch), the following brick_ctas
  // CTAs the regular bricks through tile arithmetic
  const int* brick_nb;      // [nbrick][9] first storage index of the 3x3 tiles around (and of, k = 4) the brick
  const int* irr;
  int nbrick, n_irr, brick_ctas, list_ctas;
  int n_inbox;              // cells [n_inbox, n) are the boundary cells (Neumann / Dirichlet), the only ones that read aux early
  int pf_dist;              // L2 prefetch distance in cells (one wave of resident CTAs ahead), 0 = off
  int* queue;               // pipelined sweep: this level's tile counter and CTA-done counter (both zero between launches)
};

template <int Q, bool DDF, int COLL>
struct PopLayout {
  static constexpr int G0 = Q;                                    // first plane of g
  static constexpr int L0 = (DDF ? 2 : 1) * Q;                    // first plane of lambda
  static constexpr int NPOP = L0 + (COLL == LBM_NUMEQ ? NLAMBDA : 0);
};

// Cells per thread: the fp32 weakly compressible kernels keep two consecutive Morton cells per thread (64-bit list
// loads and 64-bit stores, twice the gathers in flight per warp: with 4-byte populations one cell per thread leaves
// the memory system short of outstanding bytes, profiles/r01_ncu_uniform_f32.md); everything else one cell.
template <int Q, typename T, int COLL, bool DDF>
constexpr int cells_per_thread = (sizeof(T) == 4 && !DDF && COLL != LBM_NUMEQ && Q <= 13) ? 2 : 1;

// Resident CTAs per SM asked of ptxas (register cap = 65536 / (128 x CTAs)).  The list kernels: D2Q9 at 8 x 128 threads
// (64 registers), the fp32 D2Q13 Newton solve at 5.  The brick kernels of the polynomial models are latency-bound (one
// DRAM round trip per cell, profiles/r02_ncu_cylinder_f32.md: long_scoreboard is the top stall at 50 % of the warps), so
// they take the occupancy at which the measured throughput peaks, a few spilled bytes included (uniform 4096^2, GLUPS at
// ptxas' own choice -> here; one step further the spills win and it drops again):
//   D2Q9  fp32 10 CTAs (48 reg.)  81.2 -> 86.0    D2Q13 fp32 10 (48)  57.1 -> 62.0    D2Q21 fp32 6 (80)  34.7 -> 38.1
//   D2Q37 fp32  6 (80)  14.2 -> 16.4              D2Q13 fp64  6 (80)  31.5 -> 31.6    D2Q21 fp64 6 (80)  15.9 -> 19.4
//   D2Q37 fp64  4 (128)  7.7 ->  9.3              D2Q37 + g + sensor fp32 4 (128)  5.3 -> 8.6 (2048^2 Riemann box);
// its fp64 twin holds 148 registers of populations and loses at 3 CTAs (4.3 -> 3.8), so it stays at ptxas' 2.
template <int Q, typename T, int COLL, bool DDF, bool BRICKS = false>
constexpr int min_ctas_per_sm =
    (BRICKS && !DDF && COLL != LBM_NUMEQ) ? (Q == 9 ? (sizeof(T) == 4 ? 10 : 8) : Q == 13 ? (sizeof(T) == 4 ? 10 : 6) : Q == 21 ? 6 : (sizeof(T) == 4 ? 6 : 4))
    : (BRICKS && DDF && COLL != LBM_NUMEQ && Q == 37 && sizeof(T) == 4) ? 4
    : (Q == 9 && !DDF && COLL != LBM_NUMEQ) ? 8
    : (COLL == LBM_NUMEQ && sizeof(T) == 4 && Q == 13) ? 5 : 1;

template <typename T, int N> struct alignas(sizeof(T) * N) Vec { T v[N]; };

// Programmatic dependent launch (sm_90+): consecutive level sweeps of the schedule are chained with programmatic
// edges, so the next sweep's CTAs become resident while this sweep drains and load their static tables (type, list,
// ghost rows) before waiting for this sweep's memory to be visible.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// Newton statistics ("mean Newton iterations per update"): two 64-bit counters behind the status word,
// Newton steps (polish included) and solves; one pair of atomics per warp after a warp-level sum.
constexpr int NEWTON_COUNTER_OFFSET = 8;      // bytes from the status word
constexpr int QUEUE_COUNTER_OFFSET = 64;      // bytes from the status word: two ints per level (LBM_MAX_LEVELS x 8 = 192 bytes)
__device__ __forceinline__ void count_newton(int* status, unsigned steps, unsigned solves) {
  const unsigned m = __activemask();
  steps = __reduce_add_sync(m, steps);
  solves = __reduce_add_sync(m, solves);
  if ((threadIdx.x & 31) == __ffs(m) - 1 && solves != 0u) {
    unsigned long long* ctr = reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(status) + NEWTON_COUNTER_OFFSET);
    atomicAdd(ctr, (unsigned long long)steps);
    atomicAdd(ctr + 1, (unsigned long long)solves);
  }
}
__device__ __forceinline__ unsigned newton_steps(int it) { return (unsigned)(it < 0 ? -it - 1 : it); }

// Models whose regular interior is updated through bricks: the polynomial ones (the numerical-equilibrium kernels are
// fp64-ALU-bound, their list is 9 % of the traffic and their registers are spoken for).
template <int Q, typename T, int COLL, bool DDF>
constexpr bool has_bricks = COLL != LBM_NUMEQ;

// Regular-brick path: 64 consecutive cells = one aligned 8x8 tile of fluid cells whose pull sources are
// base[tile k] + Z-position (computed addressing in regular interiors).  Replaces (Q-1) x 4 B of
// list and the type byte per cell by 36 B per 64 cells.
// Cells of up to 104 bytes of populations (D2Q9/13 in fp64, D2Q9/13/21 in fp32): a thread owns 2 consecutive cells
// (an x-adjacent pair; 128-bit stores in fp64, 64-bit in fp32), so a brick is one warp (measured: fp64 1 -> 2 cells
// per thread +7 %; fp32 2 -> 4 cells per thread -3 %, the grid shrinks).  Wider cells (D2Q21 fp64, D2Q37, second
// distribution) keep one cell per thread (registers); a brick is then two warps.  The 9 tile bases of a brick sit in
// lanes 0-8 of each of its warps (one coalesced load) and a thread fetches by shuffle the four it can reach; tile and
// Z-position of a source follow from the thread's (x, y) by arithmetic shared between the directions (round 1 read
// them from a 64-entry table per direction and shuffled per gather: 113 of the 283 instructions per cell of the fp32
// D2Q9 kernel went into addressing, profiles/r02_ncu_cylinder_f32.md).  There is no per-cell index traffic.
// (Several bricks per warp in sequence, with the next bases prefetched, was measured
// SLOWER: uniform fp64 38.8 against 41.6 GLUPS, the 39 k-cell cavity halves -- the bricks serialise and the grid shrinks.)
template <int Q, typename T, bool DDF> constexpr int BRICK_CPT = (Q * (DDF ? 2 : 1) * (int)sizeof(T) <= 104) ? 2 : 1;
template <int Q, typename T, bool DDF> constexpr int brick_cells_per_cta = 128 * BRICK_CPT<Q, T, DDF>;

template <int Q, typename T, int COLL, bool DDF, bool SENSOR>
__device__ __forceinline__ void brick_update(const LevelArgs& a, const ModelParams& p, int block) {
  using PL = PopLayout<Q, DDF, COLL>;
  constexpr int CPT = BRICK_CPT<Q, T, DDF>;
  constexpr int TPB = 64 / CPT;                              // threads per brick: 32 or 64 (a brick never shares a warp)
  const int lane = threadIdx.x & 31;
  const int sub = threadIdx.x % TPB;                         // thread index inside its brick
  constexpr int grp = 0;                                     // lanes 0-8 of every warp hold the tile bases
  const int brick_raw = (block * 128 + threadIdx.x) / TPB;
  if (brick_raw >= a.nbrick) return;                         // whole warp beyond the last brick
  const int brick = brick_raw;
  const int m0 = sub * CPT;                                  // Z-position of this thread's first cell (x in the even bits)
  // Element index inside a buffer in 32 bits: plane * ps + cell.  lbm_grid_bind sweeps a level through bricks only where
  // NPOP * ps < 2^32 (every level of every workload here; a wider level keeps the list kernel), so an access is one
  // three-input add and one IMAD.WIDE against the buffer pointer: no 64-bit plane pointers to form or keep.
  const unsigned ps32 = (unsigned)a.ps;
  constexpr int W = Lat<Q>::t.W;
  // Tile arithmetic (the device form of grid_builder.cpp's table brick_tab, which the host verified against the list):
  // the pull source of direction i of the cell at (x, y) of the brick is cell (x - cx_i, y - cy_i) mod 8 of the tile
  // one column / row over where that difference leaves 0..7.  W <= 3 < 4, so a thread reaches at most ONE column
  // beside the centre (west if x0 < 4, else east) and one row: four tile bases per thread, a select and an add per gather.
  const int x0 = (m0 & 1) | ((m0 >> 1) & 2) | ((m0 >> 2) & 4), y0 = ((m0 >> 1) & 1) | ((m0 >> 2) & 2) | ((m0 >> 3) & 4);
  const int kx = x0 < 4 ? 0 : 2, ky = y0 < 4 ? 0 : 6;
  const int nbv = lane < 9 ? __ldg(a.brick_nb + 9ll * brick + lane) : 0;
  auto spread3 = [](int v) { return (v & 1) | ((v & 2) << 1) | ((v & 4) << 2); };
  // column terms, by d = (cell of the thread) - cx in [-W, W + CPT - 1]: Z-bits of x0 + d mod 8, and whether x0 + d left the
  // tile (never for d = 0, nor for d = 1 of an x-adjacent pair: x0 is even there)
  int colS[2 * W + CPT];
  bool colP[2 * W + CPT];
#pragma unroll
  for (int d = -W; d < W + CPT; ++d) {
    const int sx = x0 + d;
    colS[d + W] = d == 0 ? (m0 & 0x15) : (CPT == 2 && d == 1) ? (m0 & 0x15) + 1 : spread3(sx & 7);
    colP[d + W] = (d < 0 || d >= CPT) && (unsigned)sx > 7u;
  }
  pdl_wait();
  const T* __restrict__ So = (const T*)a.So;
  T* __restrict__ Sn = (T*)a.Sn;
  const int base = __shfl_sync(0xffffffffu, nbv, grp + 4);
  const int bXC = __shfl_sync(0xffffffffu, nbv, grp + 3 + kx), bCY = __shfl_sync(0xffffffffu, nbv, grp + 1 + ky);
  const int bXY = __shfl_sync(0xffffffffu, nbv, grp + kx + ky);
  // row terms, by cy: first cell of the centre-column / side-column tile of the source row + Z-bits of y0 - cy mod 8
  int rowC[2 * W + 1], rowX[2 * W + 1];
#pragma unroll
  for (int cy = -W; cy <= W; ++cy) {
    const int sy = y0 - cy;
    const int zy = cy == 0 ? (m0 & 0x2a) : spread3(sy & 7) << 1;
    const bool py = cy != 0 && (unsigned)sy > 7u;
    rowC[cy + W] = (py ? bCY : base) + zy;
    rowX[cy + W] = (py ? bXY : bXC) + zy;
  }
  T f[CPT][Q], g[CPT][Q], lam[NLAMBDA];
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int D = -Lat<Q>::t.cx[I], R = Lat<Q>::t.cy[I] + W;
    if constexpr (CPT == 2 && D == 0) {      // cx = 0: the sources of an x-adjacent pair are adjacent, one address for both
      const unsigned src = (unsigned)(rowC[R] + colS[W]);
      const T* qf = So + (src + (unsigned)I * ps32);
      f[0][I] = qf[0]; f[CPT - 1][I] = qf[1];
      if constexpr (DDF) {
        const T* qg = So + (src + (unsigned)(PL::G0 + I) * ps32);
        g[0][I] = qg[0]; g[CPT - 1][I] = qg[1];
      }
    } else {
#pragma unroll
      for (int j = 0; j < CPT; ++j) {
        const unsigned src = (unsigned)((colP[j + D + W] ? rowX[R] : rowC[R]) + colS[j + D + W]);
        f[j][I] = So[src + (unsigned)I * ps32];
        if constexpr (DDF) g[j][I] = So[src + (unsigned)(PL::G0 + I) * ps32];
      }
    }
  });
#pragma unroll
  for (int j = 0; j < CPT; ++j) {
    T rho;
    collide<Q, T, COLL, DDF, SENSOR>(p, T(a.tau), f[j], g[j], lam, rho);
    if (!(rho > T(0)) || !isfinite(rho)) atomicOr(a.status, FLAG_UNSTABLE);
  }
  const unsigned dst = (unsigned)(base + m0);
  // a brick starts at any storage index: 128-bit stores when its first cell is CPT-aligned (uniform per brick)
  if (base % CPT == 0) {
#pragma unroll
    for (int i = 0; i < Q; ++i) {
      Vec<T, CPT> o;
#pragma unroll
      for (int j = 0; j < CPT; ++j) o.v[j] = f[j][i];
      *reinterpret_cast<Vec<T, CPT>*>(Sn + (dst + (unsigned)i * ps32)) = o;
      if constexpr (DDF) {
#pragma unroll
        for (int j = 0; j < CPT; ++j) o.v[j] = g[j][i];
        *reinterpret_cast<Vec<T, CPT>*>(Sn + (dst + (unsigned)(PL::G0 + i) * ps32)) = o;
      }
    }
  } else {
#pragma unroll
    for (int i = 0; i < Q; ++i)
#pragma unroll
      for (int j = 0; j < CPT; ++j) {
        (Sn + (dst + (unsigned)i * ps32))[j] = f[j][i];
        if constexpr (DDF) (Sn + (dst + (unsigned)(PL::G0 + i) * ps32))[j] = g[j][i];
      }
  }
}

template <int Q, typename T, int COLL, bool DDF, bool SENSOR, bool BRICKS>
__global__ void __launch_bounds__(128, (min_ctas_per_sm<Q, T, COLL, DDF, BRICKS>)) sweep_kernel(const LevelArgs a, const ModelParams p) {
  using PL = PopLayout<Q, DDF, COLL>;
  constexpr bool NUMEQ = COLL == LBM_NUMEQ;
  constexpr int CPT = BRICKS ? 1 : cells_per_thread<Q, T, COLL, DDF>;
  pdl_launch_dependents();
  int c0;
  if constexpr (BRICKS) {
    static_assert(has_bricks<Q, T, COLL, DDF>, "no brick path for this model");
    if ((int)blockIdx.x >= a.list_ctas) {
      brick_update<Q, T, COLL, DDF, SENSOR>(a, p, (int)blockIdx.x - a.list_ctas);
      return;
    }
    const int t = (int)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= a.n_irr) return;
    c0 = a.irr ? a.irr[t] : t;              // irr == null: every cell of a small level through the list, one per thread
  } else {
    c0 = (blockIdx.x * blockDim.x + threadIdx.x) * CPT;
    if (c0 >= a.n) return;
  }
  const T* __restrict__ So = (const T*)a.So;
  T* __restrict__ Sn = (T*)a.Sn;
  const long long ps = a.ps;

  // ---- static tables (never written after lbm_grid_bind): cell types, links, boundary sources.  Planes are padded to
  // a multiple of 64 cells, so the vector accesses of a ragged last thread stay inside the arrays; a cell index >= n is
  // handled as a link-less fine ghost (it moves padding to padding).
  int type[CPT], side[CPT], self[CPT], nb[CPT][Q];
  {
    // every index load is issued before any is used: the type byte, the links and (boundary cells only, known from the
    // storage order) the source cell arrive together, one DRAM round trip in front of the gathers instead of two
    const Vec<unsigned char, CPT> tv = *reinterpret_cast<const Vec<unsigned char, CPT>*>(a.type + c0);
    static_for<1, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      const Vec<int, CPT> nv = *reinterpret_cast<const Vec<int, CPT>*>(a.nbr + (long long)(I - 1) * ps + c0);
#pragma unroll
      for (int j = 0; j < CPT; ++j) nb[j][I] = (c0 + j < a.n) ? nv.v[j] : LBM_LINK_NONE;
    });
    int src_cell[CPT];
#pragma unroll
    for (int j = 0; j < CPT; ++j) src_cell[j] = (c0 + j >= a.n_inbox && c0 + j < a.n) ? a.aux[c0 + j] : c0 + j;
#pragma unroll
    for (int j = 0; j < CPT; ++j) {
      const bool valid = c0 + j < a.n;
      type[j] = valid ? (tv.v[j] & TYPE_MASK) : LBM_FINE_GHOST;
      side[j] = tv.v[j] >> TYPE_SIDE_SHIFT;
      // a NEUMANN cell replicates the complete update of its source cell (reading S13)
      self[j] = (type[j] == LBM_NEUMANN) ? src_cell[j] : c0 + j;
      nb[j][0] = self[j];
    }
  }
  pdl_wait();      // from here on: data written by the previous sweeps of the stream

  // ---- step 1: gather (pull form of Eq. 31), branch-free: a wall link reads the cell's own opposite population
  // (half-way bounce-back), a NONE link the cell's own value (fine ghosts, S6; fixed up below for coarse
  // ghosts), any other link the neighbour's.
  T f[CPT][Q], g[CPT][Q], lam[CPT][NLAMBDA];
  [[maybe_unused]] unsigned n_steps = 0u, n_solves = 0u;     // Newton statistics, flushed after the stores
#pragma unroll
  for (int j = 0; j < CPT; ++j) {
    static_for<0, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      constexpr int O = Lat<Q>::t.opp[I];
      const int n = nb[j][I];
      const int src = n >= 0 ? n : self[j];
      const int comp = (n >= 0 || n == LBM_LINK_NONE) ? I : O;
      f[j][I] = So[comp * ps + src];
      if constexpr (DDF) g[j][I] = So[(PL::G0 + comp) * ps + src];
    });
  }

  // ---- next wave into L2.  A wide model keeps 8-12 warps per SM, too few to hide the two dependent DRAM round trips
  // (links, then gathers) in front of its arithmetic (profiles/r02_ncu_naca_f64.md: stall_long_scoreboard 2.5 per issue,
  // 44 % of the samples).  The CTAs that follow this one on its SM slot work pf_dist cells further along the Z-curve:
  // their link rows, and the population lines at their own indices (which hold most of their neighbours: the gathers of 128
  // consecutive Morton cells fall into the same few lines per plane), are requested now, so that their round trips end
  // in the L2.  Every line is still fetched from DRAM once; a prefetch that misses its target is only wasted.
  if (a.pf_dist > 0) {
    const long long cp = (long long)c0 + a.pf_dist;
    if (cp < a.n) {
      prefetch_l2(a.type + cp);
      static_for<1, Q>([&](auto ic) { prefetch_l2(a.nbr + (long long)(decltype(ic)::value - 1) * ps + cp); });
#pragma unroll
      for (int q = 0; q < PL::NPOP; ++q) prefetch_l2(So + q * ps + cp);
    }
  }

#pragma unroll
  for (int j = 0; j < CPT; ++j) {
    const int c = c0 + j;
    Imposed<T> imp{false, T(0), T(0), T(0), T(0)};
    if (type[j] == LBM_DIRICHLET) {
      // equilibrium Dirichlet cell: imposed (rho,u,T); rho optionally from the nearest interior cell
      const int sd = side[j];
      T rho = T(p.bc_rho[sd]);
      if (p.bc_kind[sd] == LBM_BC_DIRICHLET_EQ_RHO_EXTRAP) {
        const int s = a.aux[c];
        rho = T(0);
#pragma unroll
        for (int i = 0; i < Q; ++i) rho += So[i * ps + s];
      }
      const T Tb = (NUMEQ || DDF) ? T(p.bc_T[sd]) : T(cs2_v<Q>);
      if constexpr (NUMEQ) {
        // falls through to the one inlined Newton solver below (warm start: the cell's own stored multipliers)
        imp = Imposed<T>{true, rho, T(p.bc_ux[sd]), T(p.bc_uy[sd]), Tb};
      } else {
        T geq[Q];
        equilibrium<Q, T, COLL, DDF>(p, rho, T(p.bc_ux[sd]), T(p.bc_uy[sd]), Tb, lam[j], f[j], geq);
        if constexpr (DDF) {
#pragma unroll
          for (int i = 0; i < Q; ++i) g[j][i] = geq[i];
        }
        if (!(rho > T(0)) || !isfinite(rho)) atomicOr(a.status, FLAG_UNSTABLE);
        continue;
      }
    }

    bool special = false;     // any velocity-bounce-back or unknown link
    static_for<1, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      special |= (nb[j][I] <= LBM_LINK_VBB0) || (nb[j][I] == LBM_LINK_NONE);
    });
    if (special && !imp.on) {
      if (type[j] == LBM_COARSE_GHOST) {
        // coalescence (Eq. 4): unknown directions only, mean over the children that exist
        const int* ch = a.g_child + 4ll * a.aux[c];
        const int k0 = ch[0], k1 = ch[1], k2 = ch[2], k3 = ch[3];
        const T nf = T((k0 >= 0) + (k1 >= 0) + (k2 >= 0) + (k3 >= 0));
        const T* F = (const T*)a.fine;
        const long long fps = a.fps;
        static_for<1, Q>([&](auto ic) {
          constexpr int I = decltype(ic)::value;
          if (nb[j][I] == LBM_LINK_NONE) {
            T s = T(0);
            if (k0 >= 0) s += F[I * fps + k0];
            if (k1 >= 0) s += F[I * fps + k1];
            if (k2 >= 0) s += F[I * fps + k2];
            if (k3 >= 0) s += F[I * fps + k3];
            f[j][I] = s / nf;
            if constexpr (DDF) {
              T sg = T(0);
              if (k0 >= 0) sg += F[(PL::G0 + I) * fps + k0];
              if (k1 >= 0) sg += F[(PL::G0 + I) * fps + k1];
              if (k2 >= 0) sg += F[(PL::G0 + I) * fps + k2];
              if (k3 >= 0) sg += F[(PL::G0 + I) * fps + k3];
              g[j][I] = sg / nf;
            }
          }
        });
      }
      // velocity bounce-back (Ladd): + 2 w_i rho_w (xi_i . u_w) / c_s^2, rho_w local (S11)
      bool vbb = false;
      static_for<1, Q>([&](auto ic) { vbb |= nb[j][decltype(ic)::value] <= LBM_LINK_VBB0; });
      if (vbb) {
        T rho_w = T(0);
#pragma unroll
        for (int i = 0; i < Q; ++i) rho_w += So[i * ps + self[j]];
        static_for<1, Q>([&](auto ic) {
          constexpr int I = decltype(ic)::value;
          if (nb[j][I] <= LBM_LINK_VBB0) {
            const int sd = LBM_LINK_VBB0 - nb[j][I];
            constexpr int cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I];
            constexpr double w2 = 2.0 * Lat<Q>::t.w[I];
            const T xu = T(cx) * T(p.bc_ux[sd]) + T(cy) * T(p.bc_uy[sd]);
            f[j][I] += T(w2) * rho_w * xu / T(cs2_v<Q>);
          }
        });
      }
    }

    if (type[j] == LBM_FINE_GHOST) {
      // fine ghost cells stream without colliding; lambda stays
      if constexpr (NUMEQ) {
#pragma unroll
        for (int k = 0; k < NLAMBDA; ++k) lam[j][k] = So[(PL::L0 + k) * ps + c];
      }
      continue;
    }

    if constexpr (NUMEQ) {
      if (type[j] == LBM_COARSE_GHOST) {   // Eq. 6: warm start from the mean of the children's multipliers
        const int* ch = a.g_child + 4ll * a.aux[c];
        int nf = 0;
#pragma unroll
        for (int k = 0; k < NLAMBDA; ++k) lam[j][k] = T(0);
        for (int q = 0; q < 4; ++q) {
          const int cq = ch[q];
          if (cq < 0) continue;
          ++nf;
#pragma unroll
          for (int k = 0; k < NLAMBDA; ++k) lam[j][k] += ((const T*)a.fine)[(PL::L0 + k) * a.fps + cq];
        }
#pragma unroll
        for (int k = 0; k < NLAMBDA; ++k) lam[j][k] /= T(nf);
      } else {
#pragma unroll
        for (int k = 0; k < NLAMBDA; ++k) lam[j][k] = So[(PL::L0 + k) * ps + self[j]];
      }
    }

    // ---- pressure relaxation of the sponge (Eq. 10, "applied before the collision step" P:303; reading S24):
    // rho -> rho' = rho (1 - sigma) + sigma rho_inf at unchanged velocity and non-equilibrium part, i.e.
    // f_i += (rho'/rho - 1) f_i^eq(rho, u); a Neumann cell follows its source (S13).  Sponge cells are never in bricks.
    if constexpr (!DDF && !NUMEQ) {
      if (a.sigma != nullptr) {
        const T sg = T(a.sigma[self[j]]);
        if (sg > T(0)) {
          T r = T(0), jx = T(0), jy = T(0);
          static_for<0, Q>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            constexpr int cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I];
            r += f[j][I];
            if constexpr (cx != 0) jx += T(cx) * f[j][I];
            if constexpr (cy != 0) jy += T(cy) * f[j][I];
          });
          T ae[NA];
          aeq_moments<T>(r, jx / r, jy / r, T(0), ae);
          const T rn = r * (T(1) - sg) + sg * T(p.sponge_rho_inf);
          const T w = rn / r - T(1);
          poly_all<Q, T>(ae, [&](auto ic, T fe) { f[j][decltype(ic)::value] += w * fe; });
        }
      }
    }

    // ---- steps 2-5: moments, equilibrium, sensor, relaxation
    T rho;
    const int it = collide<Q, T, COLL, DDF, SENSOR>(p, T(a.tau), f[j], g[j], lam[j], rho, imp);
    if constexpr (NUMEQ) { n_steps += newton_steps(it); n_solves += 1u; }
    if (it < 0) atomicOr(a.status, FLAG_NEWTON);
    if (!(rho > T(0)) || !isfinite(rho)) atomicOr(a.status, FLAG_UNSTABLE);

    if (type[j] == LBM_COARSE_GHOST) {
      // uniform explosion (Eq. 5, 7): every child receives the coarse post-collision state, all directions (S8)
      const int* ch = a.g_child + 4ll * a.aux[c];
      T* F = (T*)a.fine;
      const long long fps = a.fps;
      for (int q = 0; q < 4; ++q) {
        const int cq = ch[q];
        if (cq < 0) continue;
#pragma unroll
        for (int i = 0; i < Q; ++i) F[i * fps + cq] = f[j][i];
        if constexpr (DDF) {
#pragma unroll
          for (int i = 0; i < Q; ++i) F[(PL::G0 + i) * fps + cq] = g[j][i];
        }
        if constexpr (NUMEQ) {
#pragma unroll
          for (int k = 0; k < NLAMBDA; ++k) F[(PL::L0 + k) * fps + cq] = lam[j][k];
        }
      }
    }
  }

  // ---- store (coalesced, CPT-wide: own slots of the new buffer)
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    Vec<T, CPT> o;
#pragma unroll
    for (int j = 0; j < CPT; ++j) o.v[j] = f[j][i];
    *reinterpret_cast<Vec<T, CPT>*>(Sn + i * ps + c0) = o;
  }
  if constexpr (DDF) {
#pragma unroll
    for (int i = 0; i < Q; ++i) {
      Vec<T, CPT> o;
#pragma unroll
      for (int j = 0; j < CPT; ++j) o.v[j] = g[j][i];
      *reinterpret_cast<Vec<T, CPT>*>(Sn + (PL::G0 + i) * ps + c0) = o;
    }
  }
  if constexpr (NUMEQ) {
#pragma unroll
    for (int k = 0; k < NLAMBDA; ++k) {
      Vec<T, CPT> o;
#pragma unroll
      for (int j = 0; j < CPT; ++j) o.v[j] = lam[j][k];
      *reinterpret_cast<Vec<T, CPT>*>(Sn + (PL::L0 + k) * ps + c0) = o;
    }
    count_newton(a.status, n_steps, n_solves);
  }
}

// ------------------------------------------------------------------ initialisation
struct InitArgs {
  int n;
  long long ps;
  void* S0; void* S1;
  const double* rho; const double* ux; const double* uy; const double* Tin;   // this level's slice; Tin may be null
  int* status;
};

template <int Q, typename T, int COLL, bool DDF>
__global__ void __launch_bounds__(128) init_kernel(const InitArgs a, const ModelParams p) {
  using PL = PopLayout<Q, DDF, COLL>;
  constexpr bool NUMEQ = COLL == LBM_NUMEQ;
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.n) return;
  const T r = T(a.rho[c]), vx = T(a.ux[c]), vy = T(a.uy[c]);
  const T T0 = NUMEQ ? T(p.T0) : T(cs2_v<Q>);
  const T Tc = (NUMEQ || DDF) ? (a.Tin ? T(a.Tin[c]) : T0) : T0;
  T f[Q], g[Q], lam[NLAMBDA];
  if constexpr (NUMEQ) {
    // exponents of the continuous Maxwellian as the Newton start
    lam[0] = (vx * vx + vy * vy) / (T(2) * Tc) + T(log(2.0 * 3.14159265358979323846 * (double)Tc)) - T(1);
    lam[1] = -vx / Tc; lam[2] = -vy / Tc; lam[3] = T(1) / (T(2) * Tc); lam[4] = T(0); lam[5] = T(1) / (T(2) * Tc);
    lam[6] = T(0); lam[7] = T(0);
  }
  const int it = equilibrium<Q, T, COLL, DDF>(p, r, vx, vy, Tc, lam, f, g);
  T* S0 = (T*)a.S0;
  T* S1 = (T*)a.S1;
#pragma unroll
  for (int i = 0; i < Q; ++i) { S0[i * a.ps + c] = f[i]; S1[i * a.ps + c] = f[i]; }
  if constexpr (DDF) {
#pragma unroll
    for (int i = 0; i < Q; ++i) { S0[(PL::G0 + i) * a.ps + c] = g[i]; S1[(PL::G0 + i) * a.ps + c] = g[i]; }
  }
  if constexpr (NUMEQ) {
#pragma unroll
    for (int k = 0; k < NLAMBDA; ++k) { S0[(PL::L0 + k) * a.ps + c] = lam[k]; S1[(PL::L0 + k) * a.ps + c] = lam[k]; }
  }
  if (it < 0) atomicOr(a.status, FLAG_NEWTON);
  T s = T(0);
#pragma unroll
  for (int i = 0; i < Q; ++i) s += f[i];
  if (!(s > T(0)) || !isfinite(s)) atomicOr(a.status, FLAG_UNSTABLE);
  if constexpr (NUMEQ) count_newton(a.status, newton_steps(it), 1u);
}

// Coupling of iteration 0 without streaming (listing P:202-208): per coarse ghost, coalesce the unknown
// directions from the children, collide, store in place, explode.
struct CoupleArgs {
  int ng;
  long long ps;
  void* S;                  // the coarse level's current buffer (in place)
  const int* nbr;
  const int* g_coarse;
  const int* g_child;
  void* fine; long long fps;
  double tau;
  int* status;
};

template <int Q, typename T, int COLL, bool DDF, bool SENSOR>
__global__ void __launch_bounds__(128) init_coupling_kernel(const CoupleArgs a, const ModelParams p) {
  using PL = PopLayout<Q, DDF, COLL>;
  constexpr bool NUMEQ = COLL == LBM_NUMEQ;
  T* S = (T*)a.S;
  T* fine = (T*)a.fine;
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= a.ng) return;
  const int c = a.g_coarse[q];
  const int* ch = a.g_child + 4ll * q;
  int nf = 0;
  for (int j = 0; j < 4; ++j) nf += ch[j] >= 0;
  T f[Q], g[Q], lam[NLAMBDA];
  f[0] = S[c];
  if constexpr (DDF) g[0] = S[PL::G0 * a.ps + c];
  static_for<1, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    if (a.nbr[(long long)(I - 1) * a.ps + c] == LBM_LINK_NONE) {
      T s = T(0);
      [[maybe_unused]] T sg = T(0);
      for (int j = 0; j < 4; ++j) {
        if (ch[j] < 0) continue;
        s += fine[I * a.fps + ch[j]];
        if constexpr (DDF) sg += fine[(PL::G0 + I) * a.fps + ch[j]];
      }
      f[I] = s / T(nf);
      if constexpr (DDF) g[I] = sg / T(nf);
    } else {
      f[I] = S[I * a.ps + c];
      if constexpr (DDF) g[I] = S[(PL::G0 + I) * a.ps + c];
    }
  });
  if constexpr (NUMEQ) {
#pragma unroll
    for (int k = 0; k < NLAMBDA; ++k) {
      T s = T(0);
      for (int j = 0; j < 4; ++j)
        if (ch[j] >= 0) s += fine[(PL::L0 + k) * a.fps + ch[j]];
      lam[k] = s / T(nf);
    }
  }
  T rho;
  const int it = collide<Q, T, COLL, DDF, SENSOR>(p, T(a.tau), f, g, lam, rho);
  if (it < 0) atomicOr(a.status, FLAG_NEWTON);
  if (!(rho > T(0)) || !isfinite(rho)) atomicOr(a.status, FLAG_UNSTABLE);
#pragma unroll
  for (int i = 0; i < Q; ++i) S[i * a.ps + c] = f[i];
  if constexpr (DDF) {
#pragma unroll
    for (int i = 0; i < Q; ++i) S[(PL::G0 + i) * a.ps + c] = g[i];
  }
  if constexpr (NUMEQ) {
#pragma unroll
    for (int k = 0; k < NLAMBDA; ++k) S[(PL::L0 + k) * a.ps + c] = lam[k];
  }
  for (int j = 0; j < 4; ++j) {
    const int cj = ch[j];
    if (cj < 0) continue;
#pragma unroll
    for (int i = 0; i < Q; ++i) fine[i * a.fps + cj] = f[i];
    if constexpr (DDF) {
#pragma unroll
      for (int i = 0; i < Q; ++i) fine[(PL::G0 + i) * a.fps + cj] = g[i];
    }
    if constexpr (NUMEQ) {
#pragma unroll
      for (int k = 0; k < NLAMBDA; ++k) fine[(PL::L0 + k) * a.fps + cj] = lam[k];
    }
  }
  if constexpr (NUMEQ) count_newton(a.status, newton_steps(it), 1u);
}

// rho, u, T of every cell of one level from its current populations (Eq. 51)
struct MacroArgs {
  int n;
  long long ps;
  const void* S;
  const int* cells;         // probe list (lbm_get_macroscopic_at): output t is cell cells[t]; null: output t is cell t
  double* rho; double* ux; double* uy; double* Tm;
};

template <int Q, typename T, int COLL, bool DDF>
__global__ void __launch_bounds__(128) macroscopic_kernel(const MacroArgs a, const ModelParams p) {
  using PL = PopLayout<Q, DDF, COLL>;
  constexpr bool THERMAL = (COLL == LBM_NUMEQ) || DDF;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= a.n) return;
  const int c = a.cells ? a.cells[t] : t;
  const T* S = (const T*)a.S;
  T f[Q], g[Q];
#pragma unroll
  for (int i = 0; i < Q; ++i) f[i] = S[i * a.ps + c];
  if constexpr (DDF) {
#pragma unroll
    for (int i = 0; i < Q; ++i) g[i] = S[(PL::G0 + i) * a.ps + c];
  }
  T rho, ux, uy, Tm;
  moments<Q, T, THERMAL, DDF>(p, f, g, rho, ux, uy, Tm);
  a.rho[t] = (double)rho; a.ux[t] = (double)ux; a.uy[t] = (double)uy; a.Tm[t] = (double)Tm;
}

// eps of Eq. 52 of the current (post-collision) state of every cell of one level: the refinement criterion of the
// paper's adaptive runs.  f^eq = the model's equilibrium of the cell's own moments; numerical equilibria: from the
// stored multipliers (the collision conserves the moments, so they still are this state's).
template <int Q, typename T, int COLL, bool DDF>
__device__ __forceinline__ T sensor_of_state(const ModelParams& p, const T (&f)[Q], const T (&g)[Q], const T (&lam)[NLAMBDA]) {
  constexpr bool NUMEQ = COLL == LBM_NUMEQ;
  T rho, ux, uy, Tm;
  moments<Q, T, NUMEQ || DDF, DDF>(p, f, g, rho, ux, uy, Tm);
  T feq[Q];
  if constexpr (NUMEQ) {
    if constexpr (sizeof(T) == 8) {
      NumeqExps E;
      numeq_exps(rho, lam, E);
      static_for<0, Q>([&](auto ic) { feq[decltype(ic)::value] = numeq_f<Q, decltype(ic)::value>(E); });
    } else {
      const T m0[NLAMBDA] = {};
      T sc[Q], G[NLAMBDA];
      numeq_eval<Q, T>(rho, m0, lam, feq, sc, G);
    }
  } else {
    T am[NA];
    aeq_moments<T>(rho, ux, uy, DDF ? Tm - T(cs2_v<Q>) : T(0), am);
    poly_all<Q, T>(am, [&](auto ic, T fe) { feq[decltype(ic)::value] = fe; });
  }
  T eps = T(0);
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    T den = Num<T>::abs_(feq[i]);
    if (den < Num<T>::tiny()) den = Num<T>::tiny();
    eps += Num<T>::abs_(f[i] - feq[i]) / den;
  }
  return eps / T(Q);
}

struct SensorArgs {
  int n;
  long long ps;
  const void* S;
  double* eps;
};

template <int Q, typename T, int COLL, bool DDF>
__global__ void __launch_bounds__(128) sensor_kernel(const SensorArgs a, const ModelParams p) {
  using PL = PopLayout<Q, DDF, COLL>;
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.n) return;
  const T* S = (const T*)a.S;
  T f[Q], g[Q], lam[NLAMBDA];
#pragma unroll
  for (int i = 0; i < Q; ++i) f[i] = S[i * a.ps + c];
  if constexpr (DDF) {
#pragma unroll
    for (int i = 0; i < Q; ++i) g[i] = S[(PL::G0 + i) * a.ps + c];
  }
  if constexpr (COLL == LBM_NUMEQ) {
#pragma unroll
    for (int k = 0; k < NLAMBDA; ++k) lam[k] = S[(PL::L0 + k) * a.ps + c];
  }
  a.eps[c] = (double)sensor_of_state<Q, T, COLL, DDF>(p, f, g, lam);
}

// ------------------------------------------------------------------ dispatch table entry
struct KernelSet {
  int Q, precision, collision, ddf, sensor;
  int cells_per_thread;
  const char* name;
  const void* sweep;
  const void* sweep_bricks;   // same update with compressed addressing of regular bricks, or null
  const char* bricks_name;
  int brick_cells_per_cta;
  const void* init;
  const void* couple;
  const void* macro;
  const void* sensor_field;   // eps of Eq. 52 of the stored state (lbm_get_sensor)
  // software-pipelined persistent sweep of the wide models (sweep_pipe.cuh), or null
  const void* sweep_pipe;
  const char* pipe_name;
  int pipe_tpb, pipe_smem;
  int pipe_auto;            // 1: LBM_PIPE_AUTO selects it on large levels (measured faster than one cell per thread)
  // matrix-like uniform path (matrix.cuh): even / odd AA step, initialisation, macroscopic, population export / import; or null
  const void* matrix_step[2][2];      // [one cell per thread | matrix_cpt cells per thread (nx a multiple of it)][even | odd]
  int matrix_cpt;
  const void* matrix_init;
  const void* matrix_macro;
  const void* matrix_sensor;
  const void* matrix_export;
  const void* matrix_import;
  const char* matrix_name;
};

template <int Q, typename T, int COLL, bool DDF, bool SENSOR>
KernelSet make_kernel_set(const char* name, const char* bricks_name) {
  KernelSet k;
  k.Q = Q; k.precision = (int)sizeof(T) * 8; k.collision = COLL; k.ddf = DDF; k.sensor = SENSOR;
  k.cells_per_thread = cells_per_thread<Q, T, COLL, DDF>;
  k.name = name;
  k.sweep = (const void*)&sweep_kernel<Q, T, COLL, DDF, SENSOR, false>;
  k.sweep_bricks = nullptr;
  k.bricks_name = bricks_name;
  k.brick_cells_per_cta = brick_cells_per_cta<Q, T, DDF>;
  if constexpr (has_bricks<Q, T, COLL, DDF>) k.sweep_bricks = (const void*)&sweep_kernel<Q, T, COLL, DDF, SENSOR, true>;
  k.init = (const void*)&init_kernel<Q, T, COLL, DDF>;
  k.couple = (const void*)&init_coupling_kernel<Q, T, COLL, DDF, SENSOR>;
  k.macro = (const void*)&macroscopic_kernel<Q, T, COLL, DDF>;
  k.sensor_field = (const void*)&sensor_kernel<Q, T, COLL, DDF>;
  k.sweep_pipe = nullptr; k.pipe_name = ""; k.pipe_tpb = 0; k.pipe_smem = 0; k.pipe_auto = 0;
  k.matrix_step[0][0] = k.matrix_step[0][1] = k.matrix_step[1][0] = k.matrix_step[1][1] = k.matrix_init = k.matrix_macro = k.matrix_sensor = k.matrix_export = k.matrix_import = nullptr; k.matrix_name = ""; k.matrix_cpt = 1;
  return k;
}

#define LBM_KSET(Q, T, COLL, DDF, SENSOR) \
  make_kernel_set<Q, T, COLL, DDF, SENSOR>("sweep_kernel<" #Q "," #T "," #COLL "," #DDF "," #SENSOR ",false>", \
                                           "sweep_kernel<" #Q "," #T "," #COLL "," #DDF "," #SENSOR ",true> (bricks + list)")

// defined one per lattice (sweep_q*.cu) so that the instantiations compile in parallel
int kernel_sets_q9(const KernelSet** out);
int kernel_sets_q13(const KernelSet** out);
int kernel_sets_q21(const KernelSet** out);
int kernel_sets_q37(const KernelSet** out);

}  // namespace lbm
