// lbm_api.cu -- the C ABI of include/lbm.h: device arena layout, table upload, the asynchronous
// multilevel scheduler as CUDA graphs on one stream (row a10 of SURVEY.md Sec. 8(a); listing
// P:202-215 in the canonical pull form of DESIGN.md Sec. 6), host I/O.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/lbm.h"
#include "grid.hpp"
#include "matrix.cuh"
#include "sweep.cuh"

using namespace lbm;

namespace {

constexpr int BLOCK = 128;
constexpr int64_t BRICK_MIN_LEVEL_CELLS = 1 << 18;
constexpr size_t ALIGN = 256;
static_assert(lbm::QUEUE_COUNTER_OFFSET + 8 * LBM_MAX_LEVELS <= (int)ALIGN && lbm::NEWTON_COUNTER_OFFSET + 16 <= lbm::QUEUE_COUNTER_OFFSET,
              "status word, Newton counters and the tile queues of all levels share the first ALIGN bytes of the arena");

struct DevLevel {
  int64_t n = 0, ps = 0, ng = 0;
  size_t off_type = 0, off_aux = 0, off_nbr = 0, off_gcoarse = 0, off_gchild = 0, off_S[2] = {0, 0};
  size_t off_bricks = 0, off_irr = 0, off_sigma = 0;
  double* sigma = nullptr;
  int64_t nbrick = 0, n_irr = 0;
  int* brick_nb = nullptr;
  int* irr = nullptr;
  unsigned char* type = nullptr;
  int* aux = nullptr;
  int* nbr = nullptr;
  int* g_coarse = nullptr;
  int* g_child = nullptr;
  void* S[2] = {nullptr, nullptr};
  int cur = 0;
};

template <typename T>
__global__ void export_kernel(const T* S, long long ps, int n, int comp0, int cnt, double* out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)n * cnt) return;
  const int p = (int)(t / n), c = (int)(t % n);          // coalesced reads of plane p
  out[(long long)c * cnt + p] = (double)S[(long long)(comp0 + p) * ps + c];
}

template <typename T>
__global__ void import_kernel(T* S, long long ps, int n, int comp0, int cnt, const double* in) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)n * cnt) return;
  const int p = (int)(t / n), c = (int)(t % n);
  S[(long long)(comp0 + p) * ps + c] = (T)in[(long long)c * cnt + p];
}

// ---- Re-mesh (lbm_transfer; S25 of DESIGN.md), entirely on the device: every cell of the new tree looks the old
// tree up by position -- the in-box cells of a level are stored along the Z-curve, so their Morton keys are a sorted array
// (binary search), the boundary cells are stored by (iy, ix) -- and takes: the cell stored at its own level and place (copy);
// else the nearest stored ancestor (uniform explosion, Eq. 5, 7); else the mean over the children that have data, each by copy
// or coalescence in turn (Eq. 4, 6).  A Neumann cell evaluates the rule at its source cell's place.
constexpr int TR_OFF = 1 << 20;           // boundary layers have negative coordinates
constexpr int TR_MAX_ENTRIES = 64;        // old cells under one coarsened cell (4^3)
constexpr int FLAG_EMESH = 4, FLAG_ETOODEEP = 8;

struct TrLevel {
  const unsigned long long* kin;          // Morton keys of the in-box cells, ascending = storage order
  const unsigned long long* kb;           // (iy, ix) keys of the boundary cells, ascending = storage order
  int n_in, n_b, nx, ny;
  const void* S;
  long long ps;
};
struct TrCtx { TrLevel lv[LBM_MAX_LEVELS]; int depth; };
struct TrArgs {
  int n, npop;
  long long ps;
  void* S;
  const int* ix; const int* iy; const int* aux; const unsigned char* type;
  int level;
  int* status;
};
struct TrEntry { int index, level; double weight; };

__host__ __device__ inline unsigned long long tr_spread(unsigned v) {
  unsigned long long x = v;
  x = (x | (x << 16)) & 0x0000FFFF0000FFFFull;
  x = (x | (x << 8)) & 0x00FF00FF00FF00FFull;
  x = (x | (x << 4)) & 0x0F0F0F0F0F0F0F0Full;
  x = (x | (x << 2)) & 0x3333333333333333ull;
  x = (x | (x << 1)) & 0x5555555555555555ull;
  return x;
}
__host__ __device__ inline unsigned long long tr_morton(int x, int y) { return tr_spread((unsigned)x) | (tr_spread((unsigned)y) << 1); }
__host__ __device__ inline unsigned long long tr_bkey(int x, int y) {
  return ((unsigned long long)(unsigned)(y + TR_OFF) << 32) | (unsigned)(x + TR_OFF);
}

__device__ int tr_search(const unsigned long long* k, int n, unsigned long long key) {
  int lo = 0, hi = n - 1;
  while (lo <= hi) {
    const int mid = (lo + hi) >> 1;
    const unsigned long long v = k[mid];
    if (v == key) return mid;
    if (v < key) lo = mid + 1; else hi = mid - 1;
  }
  return -1;
}

__device__ int tr_find(const TrCtx& s, int l, int x, int y) {
  if (l > s.depth) return -1;
  const TrLevel& L = s.lv[l];
  if (x >= 0 && y >= 0 && x < L.nx && y < L.ny) return tr_search(L.kin, L.n_in, tr_morton(x, y));
  const int b = tr_search(L.kb, L.n_b, tr_bkey(x, y));
  return b < 0 ? -1 : L.n_in + b;
}

// Coalescence of (l0, x0, y0), a place the old tree does not store: the old cells below it with their weights (1 / N_f per
// level crossed, N_f = the children that have data), depth first without recursion (a recursive walk would leave the stack
// size to the device limit).  Invariant: when a node is finished, the entries appended under it carry weights relative to it.
__device__ bool tr_down(const TrCtx& s, int l0, int x0, int y0, TrEntry* ent, int& n, int* status) {
  struct Frame { int l, x, y, k, start, nf; };
  Frame st[4];
  int d = 0;
  st[0] = Frame{l0, x0, y0, 0, n, 0};
  for (;;) {
    Frame& f = st[d];
    if (f.l == 0) f.k = 4;                                    // nothing below the finest level
    if (f.k == 4) {                                           // all children seen
      const bool found = f.nf > 0;
      if (found) {
        for (int e = f.start; e < n; ++e) ent[e].weight = 1.0 * ent[e].weight / (double)f.nf;
      } else {
        n = f.start;
      }
      if (d == 0) return found;
      --d;
      if (found) ++st[d].nf;
      continue;
    }
    const int k = f.k++;
    const int cl = f.l - 1, cx = 2 * f.x + (k & 1), cy = 2 * f.y + (k >> 1);
    const int c = tr_find(s, cl, cx, cy);
    if (c >= 0) {
      if (n >= TR_MAX_ENTRIES) { atomicOr(status, FLAG_ETOODEEP); return false; }
      ent[n].index = c; ent[n].level = cl; ent[n].weight = 1.0; ++n;
      ++f.nf;
    } else if (cl > 0) {
      if (d == 3) { atomicOr(status, FLAG_ETOODEEP); return false; }
      ++d;
      st[d] = Frame{cl, cx, cy, 0, n, 0};
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(128) transfer_kernel(const TrArgs a, const TrCtx s) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.n) return;
  // a Neumann cell replicates its source cell (S13): it receives what that cell receives
  const int p = (a.type[c] == LBM_NEUMANN) ? a.aux[c] : c;
  const int x = a.ix[p], y = a.iy[p], l = a.level;
  T* S = (T*)a.S;
  int sl = l, sc = tr_find(s, l, x, y);
  for (int k = 1; sc < 0 && l + k <= s.depth; ++k) {           // nearest stored ancestor (floor division: arithmetic shift)
    sc = tr_find(s, l + k, x >> k, y >> k);
    sl = l + k;
  }
  if (sc >= 0) {                                                // copy / uniform explosion: bit for bit
    const T* src = (const T*)s.lv[sl].S;
    const long long sps = s.lv[sl].ps;
    for (int q = 0; q < a.npop; ++q) S[q * a.ps + c] = src[q * sps + sc];
    return;
  }
  TrEntry ent[TR_MAX_ENTRIES];
  int n = 0;
  if (!tr_down(s, l, x, y, ent, n, a.status)) { atomicOr(a.status, FLAG_EMESH); return; }
  for (int q = 0; q < a.npop; ++q) {                            // coalescence: weights 1 / N_f per level crossed
    double acc = 0.0;
    for (int k = 0; k < n; ++k) acc += ent[k].weight * (double)((const T*)s.lv[ent[k].level].S)[q * s.lv[ent[k].level].ps + ent[k].index];
    S[q * a.ps + c] = (T)acc;
  }
}

size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

struct lbm_grid {
  HostGrid hg;
  const KernelSet* ks = nullptr;
  ModelParams mp;
  int Q = 0, npop = 0, esize = 8, depth = 0;
  std::vector<DevLevel> dl;
  int64_t n_total = 0, launches_per_coarse = 0, updates_per_coarse = 0;
  size_t arena_bytes = 0, off_status = 0, off_scratch = 0, scratch_doubles = 0;
  bool bound = false, inited = false, own_stream = false;
  int64_t brick_min_cells = BRICK_MIN_LEVEL_CELLS;   // levels below this go through the list (lbm_config.addressing: AUTO)
  bool bricks = false;                            // compressed addressing of regular bricks (off for LBM_ADDR_LIST)
  int device = -1;                                // device of the arena, selected by every entry point for its own duration
  bool pdl = true;                                // programmatic dependent launch between level sweeps (lbm_config.no_pdl)
  bool matrix = false;                            // matrix-like uniform path (matrix.cuh): one population copy, no tables on the device
  size_t off_pos = 0;
  int* d_pos = nullptr;                           // storage index -> row-major index
  int pf_dist = 0;                                // next-wave L2 prefetch distance of the one-cell-per-thread sweep of the wide models (cells)
  bool pipe = false;                              // software-pipelined persistent sweep on large levels (sweep_pipe.cuh)
  int pipe_grid = 0;                              // resident CTAs of the pipelined sweep on this device (occupancy x SMs)
  int64_t pipe_min_cells = 0;                     // levels below this keep one cell per thread
  char* arena = nullptr;
  cudaStream_t stream = nullptr;
  // level-concurrent graphs (lbm_config.concurrent_levels): the updates of levels >= 2 of a fine step are captured on a
  // side branch beside the level-0 update of the next fine step
  cudaStream_t launch_stream = nullptr;           // where enqueue_level puts its kernel (stream, or side during a capture)
  cudaStream_t side = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  bool concurrent = false;
  int* d_status = nullptr;
  double* d_scratch = nullptr;
  cudaGraphExec_t g1[2] = {nullptr, nullptr};     // one coarse step, starting parity of the coarsest level
  cudaGraphExec_t gk[2] = {nullptr, nullptr};     // K coarse steps (K even), for launch-bound small grids
  int K = 0;
  int64_t kfine = 0;                              // fine steps taken inside the current coarse step (lbm_step_fine)
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool timed = false;
};

namespace {

// Selects the grid's device for the duration of one ABI call and restores the caller's current device afterwards (the
// library links the CUDA runtime statically: the "current device" it sees is the calling thread's).
struct DeviceScope {
  int prev = -1;
  bool changed = false;
  explicit DeviceScope(int dev) {
    if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) changed = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceScope() { if (changed) cudaSetDevice(prev); }
  DeviceScope(const DeviceScope&) = delete;
  DeviceScope& operator=(const DeviceScope&) = delete;
};

#define CK(call)                                  \
  do {                                            \
    cudaError_t e_ = (call);                      \
    if (e_ != cudaSuccess) return LBM_ECUDA;      \
  } while (0)

const KernelSet* find_kernel_set(const lbm_config& c) {
  const KernelSet* sets = nullptr;
  int n = 0;
  switch (c.lattice) {
    case 9: n = kernel_sets_q9(&sets); break;
    case 13: n = kernel_sets_q13(&sets); break;
    case 21: n = kernel_sets_q21(&sets); break;
    case 37: n = kernel_sets_q37(&sets); break;
    default: return nullptr;
  }
  for (int i = 0; i < n; ++i)
    if (sets[i].precision == c.precision && sets[i].collision == c.collision && sets[i].ddf == (c.ddf != 0) &&
        sets[i].sensor == (c.sensor != 0))
      return &sets[i];
  return nullptr;
}

// n work items, `per_thread` of them per thread.  pdl: chain to the previous kernel of the stream with a programmatic
// dependent-launch edge (only for kernels that call griddepcontrol.wait before touching mutable data: the sweep).
int launch_grid(const void* fn, unsigned grid, void* a0, void* a1, cudaStream_t s, bool pdl, int smem = 0, int block = BLOCK, unsigned gridy = 1);

int launch(const void* fn, int64_t n, void* a0, void* a1, cudaStream_t s, int per_thread = 1, bool pdl = false, int smem = 0) {
  if (n <= 0) return LBM_OK;
  const int64_t threads = (n + per_thread - 1) / per_thread;
  return launch_grid(fn, (unsigned)((threads + BLOCK - 1) / BLOCK), a0, a1, s, pdl, smem);
}

int launch_grid(const void* fn, unsigned grid, void* a0, void* a1, cudaStream_t s, bool pdl, int smem, int block, unsigned gridy) {
  if (grid == 0) return LBM_OK;
  void* args[2] = {a0, a1};
  if (!pdl) {
    CK(cudaLaunchKernel(fn, dim3(grid, gridy), dim3((unsigned)block), args, (size_t)smem, s));
    return LBM_OK;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid, gridy); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = (size_t)smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  CK(cudaLaunchKernelExC(&cfg, fn, args));
  return LBM_OK;
}

MatrixArgs matrix_args(lbm_grid* g, int parity) {
  MatrixArgs a = {};
  a.nx = g->hg.lv[0].nx; a.ny = g->hg.lv[0].ny; a.n = (int)g->dl[0].n;
  a.ps = g->dl[0].ps; a.A = g->dl[0].S[0]; a.tau = g->hg.lv[0].tau; a.status = g->d_status;
  a.parity = parity; a.pos = g->d_pos;
  return a;
}

// One update of level l (old -> new buffer, coupling with level l-1 fused in), then flip its parity.
int enqueue_level(lbm_grid* g, int l, int* cur) {
  DevLevel& L = g->dl[l];
  if (g->matrix) {
    // matrix-like path: even (layout P0 -> P1) or odd (P1 -> P0) AA step in place, one thread per cell, one grid row per y
    MatrixArgs ma = matrix_args(g, cur[0]);
    const int v = (ma.nx % g->ks->matrix_cpt == 0) ? 1 : 0, cpt = v ? g->ks->matrix_cpt : 1;
    const int rc = launch_grid(g->ks->matrix_step[v][cur[0]], (unsigned)((ma.nx + BLOCK * cpt - 1) / (BLOCK * cpt)), &ma, &g->mp, g->launch_stream,
                               false, 0, BLOCK, (unsigned)ma.ny);
    if (rc == LBM_OK) cur[0] ^= 1;
    return rc;
  }
  LevelArgs a;
  a.n = (int)L.n; a.ps = L.ps;
  a.So = L.S[cur[l]]; a.Sn = L.S[1 - cur[l]];
  a.nbr = L.nbr; a.type = L.type; a.aux = L.aux; a.g_child = L.g_child;
  a.fine = l > 0 ? g->dl[l - 1].S[cur[l - 1]] : nullptr;
  a.fps = l > 0 ? g->dl[l - 1].ps : 0;
  a.tau = g->hg.lv[l].tau;
  a.status = g->d_status;
  a.sigma = L.sigma;
  a.brick_nb = L.brick_nb; a.irr = L.irr;
  a.nbrick = (int)L.nbrick; a.n_irr = (int)L.n_irr;
  a.n_inbox = (int)g->hg.lv[l].n_inbox; a.pf_dist = 0;
  a.queue = (int*)((char*)g->d_status + QUEUE_COUNTER_OFFSET) + 2 * l;
  const int64_t cells_per_cta = g->ks->brick_cells_per_cta;
  a.brick_ctas = (int)((L.nbrick * 64 + cells_per_cta - 1) / cells_per_cta);
  a.list_ctas = (int)((L.n_irr + BLOCK - 1) / BLOCK);
  // Small levels are latency-bound, not traffic-bound: they go through the list with ONE cell per thread (the list part
  // of the brick kernel with no bricks and no indirection), which gives them the most threads; measured on the 39 k-cell
  // cavity: fp64 7.4 against 6.6 GLUPS with bricks (two cells per thread).
  int rc;
  if (g->pipe && L.n >= g->pipe_min_cells) {
    // wide models, large level: persistent grid (every resident CTA slot of the device once), each thread walks over
    // n / (grid * block) cells with the next cell's gathers in flight
    const int tpb = g->ks->pipe_tpb;
    const int64_t ctas = std::min<int64_t>(g->pipe_grid, (L.n + tpb - 1) / tpb);
    // no programmatic edge into this launch: its tile queue must not be touched before the previous launch on this level has left it
    rc = launch_grid(g->ks->sweep_pipe, (unsigned)ctas, &a, &g->mp, g->launch_stream, false, g->ks->pipe_smem, tpb);
  } else if (g->bricks && L.n < g->brick_min_cells) {
    a.nbrick = 0; a.brick_ctas = 0; a.irr = nullptr; a.n_irr = (int)L.n;
    a.list_ctas = (int)((L.n + BLOCK - 1) / BLOCK);
    rc = launch_grid(g->ks->sweep_bricks, (unsigned)a.list_ctas, &a, &g->mp, g->launch_stream, g->pdl);
  } else if (g->bricks && L.nbrick > 0 && (int64_t)g->npop * L.ps < ((int64_t)1 << 32)) {
    // (brick_update indexes a buffer with 32 bits: a level of 2^32 elements or more per buffer keeps the list kernel)
    rc = launch_grid(g->ks->sweep_bricks, (unsigned)(a.list_ctas + a.brick_ctas), &a, &g->mp, g->launch_stream, g->pdl);
  } else {
    if (L.n >= 4ll * g->pf_dist) a.pf_dist = g->pf_dist;      // smaller levels live in the L2 anyway
    rc = launch(g->ks->sweep, L.n, &a, &g->mp, g->launch_stream, g->ks->cells_per_thread, g->pdl);
  }
  if (rc == LBM_OK) cur[l] ^= 1;
  return rc;
}

// Canonical (pull) form of the listing P:202-215: fine step k = 1..2^d updates level 0, then every
// level l with k = 0 mod 2^l, ascending.
int enqueue_coarse_step(lbm_grid* g, int* cur) {
  const int d = g->depth;
  // Level-concurrent variant (captures only): U(l, k) of fine step k needs U(l-1, k) (its children's values) and hands its
  // explosion to U(l-1, next), so the chain U(0..L, k) is sequential; but U(0, k+1) needs only U(1, k).  The updates of levels
  // >= 2 go to a side branch that is joined again before the next update of level 1.
  const bool conc = g->concurrent && d >= 2;
  bool forked = false;
  g->launch_stream = g->stream;
  for (int64_t k = 1; k <= ((int64_t)1 << d); ++k) {
    for (int l = 0; l <= d; ++l) {
      if (l > 0 && (k % ((int64_t)1 << l)) != 0) break;
      if (conc && l == 1 && forked) { CK(cudaStreamWaitEvent(g->stream, g->ev_join, 0)); forked = false; }
      if (conc && l == 2) {
        CK(cudaEventRecord(g->ev_fork, g->stream));
        CK(cudaStreamWaitEvent(g->side, g->ev_fork, 0));
        g->launch_stream = g->side;
      }
      int rc = enqueue_level(g, l, cur);
      if (rc) { g->launch_stream = g->stream; return rc; }
    }
    if (g->launch_stream != g->stream) {
      CK(cudaEventRecord(g->ev_join, g->side));
      forked = true;
      g->launch_stream = g->stream;
    }
  }
  if (forked) CK(cudaStreamWaitEvent(g->stream, g->ev_join, 0));
  return LBM_OK;
}

int capture(lbm_grid* g, int parity, int nsteps, cudaGraphExec_t* out) {
  std::vector<int> cur((size_t)g->depth + 1, 0);
  cur[g->depth] = parity;
  cudaGraph_t graph = nullptr;
  CK(cudaStreamBeginCapture(g->stream, cudaStreamCaptureModeThreadLocal));
  int rc = LBM_OK;
  for (int s = 0; s < nsteps && !rc; ++s) rc = enqueue_coarse_step(g, cur.data());
  cudaError_t e = cudaStreamEndCapture(g->stream, &graph);
  if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
  if (e != cudaSuccess) return LBM_ECUDA;
  e = cudaGraphInstantiate(out, graph, 0);
  cudaGraphDestroy(graph);
  return e == cudaSuccess ? LBM_OK : LBM_ECUDA;
}

int status_code(lbm_grid* g) {
  int flags = 0;
  CK(cudaMemcpyAsync(&flags, g->d_status, sizeof(int), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  if (flags & FLAG_UNSTABLE) return LBM_EUNSTABLE;
  if (flags & FLAG_NEWTON) return LBM_ENEWTON;
  return LBM_OK;
}

void release_device_objects(lbm_grid* g);

int pop_range(const lbm_grid* g, int which, int* off, int* cnt) {
  const bool ddf = g->hg.cfg.ddf != 0, numeq = g->hg.cfg.collision == LBM_NUMEQ;
  if (which == 0) { *off = 0; *cnt = g->Q; return LBM_OK; }
  if (which == 1 && ddf) { *off = g->Q; *cnt = g->Q; return LBM_OK; }
  if (which == 2 && numeq) { *off = (ddf ? 2 : 1) * g->Q; *cnt = LBM_NLAMBDA; return LBM_OK; }
  return LBM_EINVAL;
}

}  // namespace

extern "C" {

int lbm_grid_create(const lbm_config* cfg, const int64_t* split_off, const int32_t* split_xy,
                    const int64_t* solid_off, const int32_t* solid_xy, lbm_grid** out) {
  if (!cfg || !out) return LBM_EINVAL;
  *out = nullptr;
  if (cfg->precision != 64 && cfg->precision != 32) return LBM_EINVAL;
  if (cfg->collision < LBM_BGK || cfg->collision > LBM_NUMEQ) return LBM_EINVAL;
  if (cfg->collision == LBM_RR && cfg->ddf) return LBM_EINVAL;     // RR is defined for the athermal models only
  if (!(cfg->tau0 >= 0.5)) return LBM_EINVAL;
  if (cfg->addressing < LBM_ADDR_AUTO || cfg->addressing > LBM_ADDR_MATRIX) return LBM_EINVAL;
  if (cfg->addressing == LBM_ADDR_MATRIX) {
    // single-level box, weakly compressible, periodic / wall / moving-wall sides, no solids, no sponge
    if (cfg->depth != 0 || cfg->ddf || cfg->collision == LBM_NUMEQ || cfg->sponge_sigma_max != 0.0) return LBM_EINVAL;
    if (solid_off && solid_off[1] > solid_off[0]) return LBM_EINVAL;
    for (int s = 0; s < 4; ++s)
      if (cfg->bc[s] != LBM_BC_PERIODIC && cfg->bc[s] != LBM_BC_WALL && cfg->bc[s] != LBM_BC_MOVING_WALL && cfg->bc[s] != LBM_BC_INFLOW_VBB)
        return LBM_EINVAL;
  }
  if (cfg->pipeline < LBM_PIPE_AUTO || cfg->pipeline > LBM_PIPE_ALWAYS || cfg->pipe_max_ctas < 0) return LBM_EINVAL;
  // the sponge relaxes rho = p / T0: weakly compressible models only
  if (cfg->sponge_sigma_max != 0.0 && (cfg->ddf || cfg->collision == LBM_NUMEQ || !(cfg->sponge_sigma_max > 0.0) ||
                                       !(cfg->sponge_sigma_max <= 1.0) || !(cfg->sponge_r1 > cfg->sponge_r0) || !(cfg->sponge_r0 >= 0.0)))
    return LBM_EINVAL;
  // velocity bounce-back is defined for the weakly compressible models only
  for (int s = 0; s < 4; ++s)
    if ((cfg->bc[s] == LBM_BC_MOVING_WALL || cfg->bc[s] == LBM_BC_INFLOW_VBB) && (cfg->ddf || cfg->collision == LBM_NUMEQ))
      return LBM_EINVAL;
  Lattice lat;
  if (!make_lattice(cfg->lattice, &lat)) return LBM_EINVAL;
  const KernelSet* ks = find_kernel_set(*cfg);
  if (!ks) return LBM_EUNSUPPORTED;
  lbm_grid* g = new (std::nothrow) lbm_grid();
  if (!g) return LBM_ENOMEM;
  int rc = build_grid(*cfg, split_off, split_xy, solid_off, solid_xy, &g->hg);
  if (rc) { delete g; return rc; }
  try {
    g->ks = ks;
    g->Q = lat.Q;
    g->depth = cfg->depth;
    g->esize = cfg->precision / 8;
    g->npop = lat.Q * (cfg->ddf ? 2 : 1) + (cfg->collision == LBM_NUMEQ ? LBM_NLAMBDA : 0);
    g->matrix = cfg->addressing == LBM_ADDR_MATRIX;
    if (g->matrix && !ks->matrix_step[0][0]) { delete g; return LBM_EUNSUPPORTED; }
    g->bricks = ks->sweep_bricks != nullptr && cfg->addressing != LBM_ADDR_LIST && !g->matrix;
    g->brick_min_cells = !g->bricks ? INT64_MAX : cfg->addressing == LBM_ADDR_BRICKS ? 0 : BRICK_MIN_LEVEL_CELLS;
    g->concurrent = cfg->concurrent_levels != 0 && cfg->depth >= 2;
    g->pdl = cfg->no_pdl == 0 && !g->concurrent;     // programmatic edges are kept to single-stream chains
    g->pipe = ks->sweep_pipe != nullptr && (cfg->pipeline == LBM_PIPE_ALWAYS || (cfg->pipeline == LBM_PIPE_AUTO && ks->pipe_auto));
    ModelParams& mp = g->mp;
    mp.gamma = cfg->gamma; mp.sensor_A = cfg->sensor_A; mp.T0 = cfg->T0; mp.newton_tol = cfg->newton_tol;
    mp.newton_max_iter = cfg->newton_max_iter; mp.trace_eq = cfg->trace_eq;
    mp.sponge_rho_inf = cfg->sponge_rho_inf;
    for (int s = 0; s < 4; ++s) {
      mp.bc_kind[s] = cfg->bc[s];
      mp.bc_rho[s] = cfg->bc_rho[s]; mp.bc_ux[s] = cfg->bc_ux[s]; mp.bc_uy[s] = cfg->bc_uy[s]; mp.bc_T[s] = cfg->bc_T[s];
    }
    // arena layout: status word | per level: type, aux, list, ghost lists, two population buffers | scratch
    g->dl.assign((size_t)g->depth + 1, DevLevel());
    size_t off = 0;
    g->off_status = off; off += ALIGN;
    int64_t nmax = 0;
    for (int l = 0; l <= g->depth; ++l) {
      const HostLevel& H = g->hg.lv[l];
      DevLevel& L = g->dl[l];
      L.n = H.n; L.ng = H.ng;
      L.ps = (int64_t)round_up((size_t)std::max<int64_t>(H.n, 1), 64);   // planes start on 256-byte boundaries
      if (g->matrix) {
        // one population copy (AA pattern) and the storage-order map of the I/O kernels; no type, list or ghost tables
        L.nbrick = 0; L.n_irr = 0;
        L.off_S[0] = L.off_S[1] = off; off += round_up((size_t)L.ps * (size_t)g->npop * (size_t)g->esize, ALIGN);
        g->off_pos = off; off += round_up((size_t)L.ps * 4, ALIGN);
      } else {
        L.off_type = off; off += round_up((size_t)L.ps, ALIGN);
        L.off_aux = off; off += round_up((size_t)L.ps * 4, ALIGN);
        L.off_nbr = off; off += round_up((size_t)L.ps * 4 * (size_t)(g->Q - 1), ALIGN);
        L.off_gcoarse = off; off += round_up((size_t)std::max<int64_t>(H.ng, 1) * 4, ALIGN);
        L.off_gchild = off; off += round_up((size_t)std::max<int64_t>(H.ng, 1) * 16, ALIGN);
        L.nbrick = H.nbrick; L.n_irr = (int64_t)H.irr.size();
        L.off_bricks = off; off += round_up((size_t)std::max<int64_t>(H.nbrick, 1) * 36, ALIGN);
        L.off_irr = off; off += round_up((size_t)std::max<int64_t>(L.n_irr, 1) * 4, ALIGN);
        L.off_sigma = off; off += round_up(H.sigma.size() * 8, ALIGN);
        for (int b = 0; b < 2; ++b) { L.off_S[b] = off; off += round_up((size_t)L.ps * (size_t)g->npop * (size_t)g->esize, ALIGN); }
      }
      g->n_total += H.n;
      nmax = std::max(nmax, H.n);
      g->updates_per_coarse += H.n << (g->depth - l);
      g->launches_per_coarse += (H.n > 0 ? 1 : 0) * ((int64_t)1 << (g->depth - l));
    }
    g->scratch_doubles = (size_t)std::max<int64_t>(4 * g->n_total, nmax * std::max(g->Q, LBM_NLAMBDA)) + 8;
    g->off_scratch = off; off += round_up(g->scratch_doubles * 8, ALIGN);
    g->arena_bytes = off;
  } catch (const std::bad_alloc&) {
    delete g;
    return LBM_ENOMEM;
  }
  *out = g;
  return LBM_OK;
}

void lbm_destroy(lbm_grid* g) {
  if (!g) return;
  if (g->bound) {
    DeviceScope dev(g->device);
    cudaStreamSynchronize(g->stream);
    release_device_objects(g);
  }
  delete g;
}

int lbm_grid_query(const lbm_grid* g, lbm_grid_info* o) {
  if (!g || !o) return LBM_EINVAL;
  memset(o, 0, sizeof(*o));
  o->depth = g->depth; o->Q = g->Q; o->W = g->hg.lat.W; o->npop = g->npop; o->precision = g->hg.cfg.precision;
  for (int l = 0; l <= g->depth; ++l) {
    const HostLevel& H = g->hg.lv[l];
    o->n_cells[l] = H.n; o->n_inbox[l] = H.n_inbox; o->n_coarse_ghosts[l] = H.ng; o->n_fine_ghosts[l] = H.n_fine_ghost;
    o->tau[l] = H.tau;
    o->n_bricks[l] = H.nbrick;
  }
  o->brick_min_level_cells = g->brick_min_cells;
  o->n_total = g->n_total;
  o->updates_per_coarse_step = g->updates_per_coarse;
  o->launches_per_coarse_step = g->launches_per_coarse;
  o->arena_bytes = g->arena_bytes;
  return LBM_OK;
}

int lbm_get_cells(const lbm_grid* g, int l, int32_t* ix, int32_t* iy, int32_t* type, int32_t* aux) {
  if (!g || l < 0 || l > g->depth) return LBM_EINVAL;
  const HostLevel& H = g->hg.lv[l];
  for (int64_t c = 0; c < H.n; ++c) {
    if (ix) ix[c] = H.ix[c];
    if (iy) iy[c] = H.iy[c];
    if (type) type[c] = H.type[c];
    if (aux) aux[c] = H.aux[c];
  }
  return LBM_OK;
}

int lbm_get_nbr(const lbm_grid* g, int l, int32_t* nbr) {
  if (!g || !nbr || l < 0 || l > g->depth) return LBM_EINVAL;
  const HostLevel& H = g->hg.lv[l];
  const int Q = g->Q;
  for (int i = 1; i < Q; ++i)
    for (int64_t c = 0; c < H.n; ++c) nbr[c * (Q - 1) + i - 1] = H.nbr[(size_t)(i - 1) * H.n + c];
  return LBM_OK;
}

int lbm_get_ghosts(const lbm_grid* g, int l, int32_t* coarse, int32_t* child, uint64_t* mask) {
  if (!g || l < 1 || l > g->depth) return LBM_EINVAL;
  const HostLevel& H = g->hg.lv[l];
  if (coarse) memcpy(coarse, H.g_coarse.data(), sizeof(int32_t) * (size_t)H.ng);
  if (child) memcpy(child, H.g_child.data(), sizeof(int32_t) * (size_t)(4 * H.ng));
  if (mask) memcpy(mask, H.g_mask.data(), sizeof(uint64_t) * (size_t)H.ng);
  return LBM_OK;
}

int lbm_get_bricks(const lbm_grid* g, int l, int32_t* tiles9, uint16_t* table) {
  if (!g || l < 0 || l > g->depth) return LBM_EINVAL;
  const HostLevel& H = g->hg.lv[l];
  if (tiles9 && H.nbrick > 0) memcpy(tiles9, H.brick_nb.data(), sizeof(int32_t) * (size_t)(9 * H.nbrick));
  if (table) memcpy(table, g->hg.brick_tab.data(), sizeof(uint16_t) * g->hg.brick_tab.size());
  return LBM_OK;
}

int lbm_get_sponge(const lbm_grid* g, int l, double* sigma) {
  if (!g || !sigma || l < 0 || l > g->depth) return LBM_EINVAL;
  const HostLevel& H = g->hg.lv[l];
  for (int64_t c = 0; c < H.n; ++c) sigma[c] = H.sigma.empty() ? 0.0 : H.sigma[(size_t)c];
  return LBM_OK;
}

int lbm_get_schedule(const lbm_grid* g, int32_t* k_of, int32_t* level_of, int cap) {
  if (!g) return LBM_EINVAL;
  int n = 0;
  for (int64_t k = 1; k <= ((int64_t)1 << g->depth); ++k)
    for (int l = 0; l <= g->depth; ++l) {
      if (l > 0 && (k % ((int64_t)1 << l)) != 0) break;
      if (n < cap) {
        if (k_of) k_of[n] = (int32_t)k;
        if (level_of) level_of[n] = l;
      }
      ++n;
    }
  return n;
}

}  // extern "C"

namespace {

void release_device_objects(lbm_grid* g) {
  for (int p = 0; p < 2; ++p) {
    if (g->g1[p]) { cudaGraphExecDestroy(g->g1[p]); g->g1[p] = nullptr; }
    if (g->gk[p]) { cudaGraphExecDestroy(g->gk[p]); g->gk[p] = nullptr; }
  }
  if (g->ev0) { cudaEventDestroy(g->ev0); g->ev0 = nullptr; }
  if (g->ev1) { cudaEventDestroy(g->ev1); g->ev1 = nullptr; }
  if (g->ev_fork) { cudaEventDestroy(g->ev_fork); g->ev_fork = nullptr; }
  if (g->ev_join) { cudaEventDestroy(g->ev_join); g->ev_join = nullptr; }
  if (g->side) { cudaStreamDestroy(g->side); g->side = nullptr; }
  if (g->own_stream && g->stream) cudaStreamDestroy(g->stream);
  g->stream = nullptr; g->own_stream = false;
}

int bind_impl(lbm_grid* g, void* dev_arena, void* cuda_stream) {
  g->arena = (char*)dev_arena;
  if (cuda_stream) {
    g->stream = (cudaStream_t)cuda_stream;
  } else {
    CK(cudaStreamCreateWithFlags(&g->stream, cudaStreamNonBlocking));
    g->own_stream = true;
  }
  g->d_status = (int*)(g->arena + g->off_status);
  g->d_scratch = (double*)(g->arena + g->off_scratch);
  CK(cudaMemsetAsync(g->d_status, 0, ALIGN, g->stream));
  const int Q = g->Q;
  std::vector<unsigned char> tbytes;
  if (g->matrix) {
    const HostLevel& H = g->hg.lv[0];
    DevLevel& L = g->dl[0];
    if (H.ny > 65535) return LBM_EINVAL;            // one grid row per y
    L.S[0] = L.S[1] = g->arena + L.off_S[0];
    L.cur = 0;
    g->d_pos = (int*)(g->arena + g->off_pos);
    std::vector<int32_t> pos((size_t)H.n);
    for (int64_t c = 0; c < H.n; ++c) pos[(size_t)c] = H.iy[c] * H.nx + H.ix[c];
    CK(cudaMemcpyAsync(g->d_pos, pos.data(), (size_t)H.n * 4, cudaMemcpyHostToDevice, g->stream));
    CK(cudaMemsetAsync(L.S[0], 0, (size_t)L.ps * g->npop * g->esize, g->stream));
    CK(cudaStreamSynchronize(g->stream));
  }
  for (int l = 0; l <= g->depth && !g->matrix; ++l) {
    const HostLevel& H = g->hg.lv[l];
    DevLevel& L = g->dl[l];
    L.type = (unsigned char*)(g->arena + L.off_type);
    L.aux = (int*)(g->arena + L.off_aux);
    L.nbr = (int*)(g->arena + L.off_nbr);
    L.g_coarse = (int*)(g->arena + L.off_gcoarse);
    L.g_child = (int*)(g->arena + L.off_gchild);
    for (int b = 0; b < 2; ++b) L.S[b] = g->arena + L.off_S[b];
    L.cur = 0;
    if (H.n == 0) continue;
    tbytes.resize((size_t)H.n);
    for (int64_t c = 0; c < H.n; ++c) tbytes[c] = (unsigned char)(H.type[c] | (H.side[c] << TYPE_SIDE_SHIFT));
    CK(cudaMemcpyAsync(L.type, tbytes.data(), (size_t)H.n, cudaMemcpyHostToDevice, g->stream));
    CK(cudaStreamSynchronize(g->stream));   // tbytes is reused per level
    CK(cudaMemcpyAsync(L.aux, H.aux.data(), (size_t)H.n * 4, cudaMemcpyHostToDevice, g->stream));
    CK(cudaMemcpy2DAsync(L.nbr, (size_t)L.ps * 4, H.nbr.data(), (size_t)H.n * 4, (size_t)H.n * 4, (size_t)(Q - 1),
                         cudaMemcpyHostToDevice, g->stream));
    L.brick_nb = (int*)(g->arena + L.off_bricks);
    L.irr = (int*)(g->arena + L.off_irr);
    if (H.nbrick > 0) CK(cudaMemcpyAsync(L.brick_nb, H.brick_nb.data(), (size_t)H.nbrick * 36, cudaMemcpyHostToDevice, g->stream));
    if (!H.irr.empty()) CK(cudaMemcpyAsync(L.irr, H.irr.data(), H.irr.size() * 4, cudaMemcpyHostToDevice, g->stream));
    L.sigma = H.sigma.empty() ? nullptr : (double*)(g->arena + L.off_sigma);
    if (L.sigma) CK(cudaMemcpyAsync(L.sigma, H.sigma.data(), H.sigma.size() * 8, cudaMemcpyHostToDevice, g->stream));
    if (H.ng > 0) {
      CK(cudaMemcpyAsync(L.g_coarse, H.g_coarse.data(), (size_t)H.ng * 4, cudaMemcpyHostToDevice, g->stream));
      CK(cudaMemcpyAsync(L.g_child, H.g_child.data(), (size_t)H.ng * 16, cudaMemcpyHostToDevice, g->stream));
    }
    // padding of the population planes is never read by a valid link; zero it once so that exports are clean
    for (int b = 0; b < 2; ++b) CK(cudaMemsetAsync(L.S[b], 0, (size_t)L.ps * g->npop * g->esize, g->stream));
  }
  CK(cudaStreamSynchronize(g->stream));
  CK(cudaEventCreate(&g->ev0));
  CK(cudaEventCreate(&g->ev1));
  g->launch_stream = g->stream;
  if (g->concurrent) {
    CK(cudaStreamCreateWithFlags(&g->side, cudaStreamNonBlocking));
    CK(cudaEventCreateWithFlags(&g->ev_fork, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&g->ev_join, cudaEventDisableTiming));
  }
  if ((g->hg.cfg.ddf || g->hg.cfg.collision == LBM_NUMEQ) && g->hg.cfg.no_prefetch == 0) {
    // wide models: distance of the next-wave L2 prefetch = the cells one wave of resident CTAs covers
    int per_sm = 0, sms = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, g->ks->sweep, BLOCK, 0));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, g->device));
    g->pf_dist = per_sm * sms * BLOCK * g->ks->cells_per_thread;
  }
  if (g->pipe) {
    // the pipelined sweep stages two cells per thread in shared memory (opt-in above 48 KB) and is launched as ONE wave:
    // grid = resident CTAs per SM (registers and shared memory decide) x SMs of this device
    int per_sm = 0, sms = 0;
    CK(cudaFuncSetAttribute(g->ks->sweep_pipe, cudaFuncAttributeMaxDynamicSharedMemorySize, g->ks->pipe_smem));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, g->ks->sweep_pipe, g->ks->pipe_tpb, (size_t)g->ks->pipe_smem));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, g->device));
    if (per_sm < 1 || sms < 1) return LBM_ECUDA;
    g->pipe_grid = per_sm * sms;
    if (g->hg.cfg.pipe_max_ctas > 0) g->pipe_grid = std::min(g->pipe_grid, g->hg.cfg.pipe_max_ctas);
    // a level must give every thread at least two cells for the prefetch to overlap anything
    g->pipe_min_cells = g->hg.cfg.pipeline == LBM_PIPE_ALWAYS ? 0 : 2ll * g->pipe_grid * g->ks->pipe_tpb;
  }
  // graphs (one coarse step from either parity of the coarsest level; K steps for launch-bound grids) are captured on
  // first use by lbm_step and dropped when a parameter baked into their kernel arguments changes
  g->K = 0;
  if (g->launches_per_coarse > 0 && g->launches_per_coarse <= 32) {
    int K = (int)(128 / g->launches_per_coarse);
    K -= K & 1;
    if (K >= 2) g->K = K;
  }
  return LBM_OK;
}

}  // namespace

extern "C" {

int lbm_grid_bind(lbm_grid* g, void* dev_arena, size_t nbytes, void* cuda_stream) {
  if (!g || !dev_arena) return LBM_EINVAL;
  if (g->bound) return LBM_ESTATE;
  if (nbytes < g->arena_bytes || ((uintptr_t)dev_arena % ALIGN) != 0) return LBM_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return LBM_ECUDA;   // no CPU fallback
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, dev_arena) != cudaSuccess) { cudaGetLastError(); return LBM_ECUDA; }
  if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) return LBM_EINVAL;   // host pointers are not an arena
  g->device = at.device;
  DeviceScope dev(g->device);
  const int rc = bind_impl(g, dev_arena, cuda_stream);
  if (rc != LBM_OK) {            // nothing stays attached: the stream and events created so far are released
    release_device_objects(g);
    g->arena = nullptr; g->device = -1;
    return rc;
  }
  g->bound = true;
  return LBM_OK;
}

int lbm_init_fields(lbm_grid* g, const double* rho, const double* ux, const double* uy, const double* T) {
  if (!g || !rho || !ux || !uy) return LBM_EINVAL;
  if (!g->bound) return LBM_ESTATE;
  DeviceScope dev(g->device);
  g->inited = false;
  const size_t N = (size_t)g->n_total;
  double* d_rho = g->d_scratch;
  double* d_ux = d_rho + N;
  double* d_uy = d_ux + N;
  double* d_T = d_uy + N;
  CK(cudaMemsetAsync(g->d_status, 0, sizeof(int), g->stream));
  CK(cudaMemcpyAsync(d_rho, rho, N * 8, cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(d_ux, ux, N * 8, cudaMemcpyHostToDevice, g->stream));
  CK(cudaMemcpyAsync(d_uy, uy, N * 8, cudaMemcpyHostToDevice, g->stream));
  if (T) CK(cudaMemcpyAsync(d_T, T, N * 8, cudaMemcpyHostToDevice, g->stream));
  if (g->matrix) {
    MatrixArgs ma = matrix_args(g, 0);
    ma.rho = d_rho; ma.ux = d_ux; ma.uy = d_uy;
    int rc = launch(g->ks->matrix_init, g->dl[0].n, &ma, &g->mp, g->stream);
    if (rc) return rc;
    g->dl[0].cur = 0;
    g->inited = true; g->timed = false; g->kfine = 0;
    return status_code(g);
  }
  int64_t base = 0;
  for (int l = 0; l <= g->depth; ++l) {
    DevLevel& L = g->dl[l];
    InitArgs a;
    a.n = (int)L.n; a.ps = L.ps; a.S0 = L.S[0]; a.S1 = L.S[1];
    a.rho = d_rho + base; a.ux = d_ux + base; a.uy = d_uy + base; a.Tin = T ? d_T + base : nullptr;
    a.status = g->d_status;
    int rc = launch(g->ks->init, L.n, &a, &g->mp, g->stream);
    if (rc) return rc;
    L.cur = 0;
    base += L.n;
  }
  // coupling of iteration 0 (listing P:202-208), coarsest interface first
  for (int l = g->depth; l >= 1; --l) {
    DevLevel& L = g->dl[l];
    if (L.ng == 0) continue;
    CoupleArgs a;
    a.ng = (int)L.ng; a.ps = L.ps; a.S = L.S[0]; a.nbr = L.nbr; a.g_coarse = L.g_coarse; a.g_child = L.g_child;
    a.fine = g->dl[l - 1].S[0]; a.fps = g->dl[l - 1].ps; a.tau = g->hg.lv[l].tau; a.status = g->d_status;
    int rc = launch(g->ks->couple, L.ng, &a, &g->mp, g->stream);
    if (rc) return rc;
  }
  g->inited = true;
  g->timed = false;
  g->kfine = 0;
  return status_code(g);
}

int lbm_step_fine(lbm_grid* g, int n) {
  if (!g || n < 0) return LBM_EINVAL;
  if (!g->bound || !g->inited) return LBM_ESTATE;
  DeviceScope dev(g->device);
  const int d = g->depth;
  std::vector<int> cur((size_t)d + 1);
  for (int l = 0; l <= d; ++l) cur[l] = g->dl[l].cur;
  // a launch that fails in the middle of a fine step leaves some levels advanced and others not: the grid is then marked
  // uninitialised (every compute call returns LBM_ESTATE until the next lbm_init_fields) instead of running on with
  // buffer parities that no longer describe the device state
  g->inited = false;
  g->launch_stream = g->stream;
  CK(cudaEventRecord(g->ev0, g->stream));
  for (int s = 0; s < n; ++s) {
    const int64_t k = g->kfine + 1;               // schedule of DESIGN.md Sec. 6 rule 9 at fine step k
    for (int l = 0; l <= d; ++l) {
      if (l > 0 && (k % ((int64_t)1 << l)) != 0) break;
      int rc = enqueue_level(g, l, cur.data());
      if (rc) return rc;
    }
    g->kfine = k % ((int64_t)1 << d);
    for (int l = 0; l <= d; ++l) g->dl[l].cur = cur[l];
  }
  CK(cudaEventRecord(g->ev1, g->stream));
  g->inited = true;
  g->timed = true;
  return LBM_OK;
}

int lbm_step(lbm_grid* g, int n) {
  if (!g || n < 0) return LBM_EINVAL;
  if (!g->bound || !g->inited) return LBM_ESTATE;
  if (g->kfine != 0) return LBM_ESTATE;           // graphs start at a coarse-step boundary
  DeviceScope dev(g->device);
  int& p = g->dl[g->depth].cur;
  // capture what this call needs before the timed region starts: n = nk launches of the K-step graph (parity kept) and
  // r single steps that alternate the parity
  const int nk = g->K >= 2 ? n / g->K : 0, r = n - nk * g->K;
  if (nk > 0 && !g->gk[p]) { int rc = capture(g, p, g->K, &g->gk[p]); if (rc) return rc; }
  if (r >= 1 && !g->g1[p]) { int rc = capture(g, p, 1, &g->g1[p]); if (rc) return rc; }
  if (r >= 2 && !g->g1[p ^ 1]) { int rc = capture(g, p ^ 1, 1, &g->g1[p ^ 1]); if (rc) return rc; }
  g->inited = false;                                // see lbm_step_fine: restored once everything is enqueued
  CK(cudaEventRecord(g->ev0, g->stream));
  while (n > 0) {
    if (g->K >= 2 && n >= g->K) {
      CK(cudaGraphLaunch(g->gk[p], g->stream));     // K even: parity unchanged
      n -= g->K;
    } else {
      CK(cudaGraphLaunch(g->g1[p], g->stream));
      p ^= 1;                                       // one coarse step flips the coarsest level once, every other level an even number of times
      n -= 1;
    }
  }
  CK(cudaEventRecord(g->ev1, g->stream));
  g->inited = true;
  g->timed = true;
  return LBM_OK;
}

namespace {
void drop_graphs(lbm_grid* g) {
  if (!g->bound) return;
  DeviceScope dev(g->device);
  cudaStreamSynchronize(g->stream);
  for (int p = 0; p < 2; ++p) {
    if (g->g1[p]) { cudaGraphExecDestroy(g->g1[p]); g->g1[p] = nullptr; }
    if (g->gk[p]) { cudaGraphExecDestroy(g->gk[p]); g->gk[p] = nullptr; }
  }
}
}  // namespace

int lbm_set_relaxation(lbm_grid* g, double tau0) {
  if (!g || !(tau0 >= 0.5)) return LBM_EINVAL;
  g->hg.cfg.tau0 = tau0;
  for (int l = 0; l <= g->depth; ++l) g->hg.lv[l].tau = 0.5 + (tau0 - 0.5) / (double)((int64_t)1 << l);   // Eq. 3 (S3)
  drop_graphs(g);
  return LBM_OK;
}

int lbm_set_boundary_state(lbm_grid* g, int side, double rho, double ux, double uy, double T) {
  if (!g || side < 0 || side > 3) return LBM_EINVAL;
  // matrix-like path: Ladd's term of the OLD wall velocity is folded into the stored wall slots (matrix.cuh); the state is taken
  // out with the old parameters and put back with the new ones, so that the next pull sees the new wall velocity as the list
  // path (and the oracle) would
  const bool rebake = g->matrix && g->bound && g->inited;
  if (rebake) {
    DeviceScope dev(g->device);
    MatrixArgs ma = matrix_args(g, g->dl[0].cur);
    ma.pops = g->d_scratch;
    int rc = launch(g->ks->matrix_export, g->dl[0].n, &ma, &g->mp, g->stream);
    if (rc) return rc;
    CK(cudaStreamSynchronize(g->stream));          // the kernel read g->mp by value at launch; be explicit all the same
  }
  g->hg.cfg.bc_rho[side] = rho; g->hg.cfg.bc_ux[side] = ux; g->hg.cfg.bc_uy[side] = uy; g->hg.cfg.bc_T[side] = T;
  g->mp.bc_rho[side] = rho; g->mp.bc_ux[side] = ux; g->mp.bc_uy[side] = uy; g->mp.bc_T[side] = T;
  drop_graphs(g);
  if (rebake) {
    DeviceScope dev(g->device);
    MatrixArgs ma = matrix_args(g, g->dl[0].cur);
    ma.pops = g->d_scratch;
    int rc = launch(g->ks->matrix_import, g->dl[0].n, &ma, &g->mp, g->stream);
    if (rc) return rc;
  }
  return LBM_OK;
}

int lbm_transfer(lbm_grid* dst, lbm_grid* src) {
  if (!dst || !src || dst == src) return LBM_EINVAL;
  if (!dst->bound || !src->bound || !src->inited) return LBM_ESTATE;
  if (src->kfine != 0) return LBM_ESTATE;
  if (dst->matrix || src->matrix || dst->device != src->device) return LBM_EINVAL;
  const lbm_config &a = dst->hg.cfg, &b = src->hg.cfg;
  if (a.lattice != b.lattice || a.precision != b.precision || a.collision != b.collision || (a.ddf != 0) != (b.ddf != 0)) return LBM_EINVAL;
  if (src->hg.lat.Q != dst->hg.lat.Q) return LBM_EINVAL;
  if (((int64_t)b.nx_coarse << src->depth) != ((int64_t)a.nx_coarse << dst->depth) ||
      ((int64_t)b.ny_coarse << src->depth) != ((int64_t)a.ny_coarse << dst->depth))
    return LBM_EINVAL;
  DeviceScope dev(dst->device);
  CK(cudaStreamSynchronize(src->stream));
  dst->inited = false;
  CK(cudaMemsetAsync(dst->d_status, 0, sizeof(int), dst->stream));
  // position keys of the old tree -> src's scratch area (8 bytes per cell), level after level
  TrCtx ctx = {};
  ctx.depth = src->depth;
  {
    std::vector<unsigned long long> keys((size_t)src->n_total);
    size_t base = 0;
    for (int l = 0; l <= src->depth; ++l) {
      const HostLevel& H = src->hg.lv[l];
      for (int64_t c = 0; c < H.n; ++c)
        keys[base + (size_t)c] = c < H.n_inbox ? tr_morton(H.ix[c], H.iy[c]) : tr_bkey(H.ix[c], H.iy[c]);
      for (int64_t c = 1; c < H.n; ++c)       // the storage order IS the key order (DESIGN.md Sec. 6 rule 6): what the search relies on
        if (c != H.n_inbox && keys[base + (size_t)c] <= keys[base + (size_t)c - 1]) return LBM_EINVAL;
      TrLevel& L = ctx.lv[l];
      L.kin = (const unsigned long long*)src->d_scratch + base;
      L.kb = L.kin + H.n_inbox;
      L.n_in = (int)H.n_inbox; L.n_b = (int)(H.n - H.n_inbox); L.nx = H.nx; L.ny = H.ny;
      L.S = src->dl[l].S[src->dl[l].cur]; L.ps = src->dl[l].ps;
      base += (size_t)H.n;
    }
    if (keys.size() > src->scratch_doubles) return LBM_ENOMEM;
    CK(cudaMemcpyAsync(src->d_scratch, keys.data(), keys.size() * 8, cudaMemcpyHostToDevice, dst->stream));
    CK(cudaStreamSynchronize(dst->stream));
  }
  // positions, types and sources of the new tree -> dst's scratch area (13 bytes per cell), then one launch per level
  {
    const size_t N = (size_t)dst->n_total;
    if (4 * N * 4 > dst->scratch_doubles * 8) return LBM_ENOMEM;
    std::vector<int32_t> hix(N), hiy(N), haux(N);
    std::vector<unsigned char> hty(N);
    size_t base = 0;
    for (int l = 0; l <= dst->depth; ++l) {
      const HostLevel& H = dst->hg.lv[l];
      for (int64_t c = 0; c < H.n; ++c) {
        hix[base + (size_t)c] = H.ix[c]; hiy[base + (size_t)c] = H.iy[c]; haux[base + (size_t)c] = H.aux[c];
        hty[base + (size_t)c] = H.type[c];
        if (H.type[c] == LBM_NEUMANN && (H.aux[c] < 0 || H.aux[c] >= H.n)) return LBM_EMESH;
      }
      base += (size_t)H.n;
    }
    int* d_ix = (int*)dst->d_scratch;
    int* d_iy = d_ix + N;
    int* d_aux = d_iy + N;
    unsigned char* d_ty = (unsigned char*)(d_aux + N);
    CK(cudaMemcpyAsync(d_ix, hix.data(), N * 4, cudaMemcpyHostToDevice, dst->stream));
    CK(cudaMemcpyAsync(d_iy, hiy.data(), N * 4, cudaMemcpyHostToDevice, dst->stream));
    CK(cudaMemcpyAsync(d_aux, haux.data(), N * 4, cudaMemcpyHostToDevice, dst->stream));
    CK(cudaMemcpyAsync(d_ty, hty.data(), N, cudaMemcpyHostToDevice, dst->stream));
    base = 0;
    for (int l = 0; l <= dst->depth; ++l) {
      DevLevel& L = dst->dl[l];
      L.cur = 0;
      TrArgs ta = {};
      ta.n = (int)L.n; ta.npop = dst->npop; ta.ps = L.ps; ta.S = L.S[0];
      ta.ix = d_ix + base; ta.iy = d_iy + base; ta.aux = d_aux + base; ta.type = d_ty + base;
      ta.level = l; ta.status = dst->d_status;
      const unsigned grid = (unsigned)((L.n + BLOCK - 1) / BLOCK);
      if (grid > 0) {
        if (dst->esize == 8) transfer_kernel<double><<<grid, BLOCK, 0, dst->stream>>>(ta, ctx);
        else transfer_kernel<float><<<grid, BLOCK, 0, dst->stream>>>(ta, ctx);
        CK(cudaGetLastError());
      }
      base += (size_t)L.n;
    }
    int flags = 0;
    CK(cudaMemcpyAsync(&flags, dst->d_status, sizeof(int), cudaMemcpyDeviceToHost, dst->stream));
    CK(cudaStreamSynchronize(dst->stream));                    // the host vectors above live until here
    CK(cudaMemsetAsync(dst->d_status, 0, sizeof(int), dst->stream));
    if (flags & FLAG_EMESH) return LBM_EMESH;                 // the old tree has no data under a cell of the new one
    if (flags & FLAG_ETOODEEP) return LBM_EINVAL;             // a cell coarsened over more than three levels at once
  }
  dst->inited = true; dst->timed = false; dst->kfine = 0;
  return LBM_OK;
}

int lbm_sync(lbm_grid* g) {
  if (!g) return LBM_EINVAL;
  if (!g->bound) return LBM_ESTATE;
  DeviceScope dev(g->device);
  return status_code(g);
}

double lbm_last_step_ms(lbm_grid* g) {
  if (!g) return (double)LBM_EINVAL;
  if (!g->bound || !g->timed) return (double)LBM_ESTATE;
  DeviceScope dev(g->device);
  if (cudaEventSynchronize(g->ev1) != cudaSuccess) return (double)LBM_ECUDA;
  float ms = 0.f;
  if (cudaEventElapsedTime(&ms, g->ev0, g->ev1) != cudaSuccess) return (double)LBM_ECUDA;
  return (double)ms;
}

int lbm_supported_model(int index, lbm_config* out) {
  if (index < 0 || !out) return LBM_EINVAL;
  const KernelSet* sets = nullptr;
  int base = 0;
  for (int lat = 0; lat < 4; ++lat) {
    const int n = lat == 0 ? kernel_sets_q9(&sets) : lat == 1 ? kernel_sets_q13(&sets) : lat == 2 ? kernel_sets_q21(&sets) : kernel_sets_q37(&sets);
    if (index < base + n) {
      const KernelSet& k = sets[index - base];
      memset(out, 0, sizeof(*out));
      out->lattice = k.Q; out->precision = k.precision; out->collision = k.collision; out->ddf = k.ddf; out->sensor = k.sensor;
      return LBM_OK;
    }
    base += n;
  }
  return LBM_EINVAL;
}

int lbm_newton_iterations(lbm_grid* g, int64_t* iterations, int64_t* solves) {
  if (!g) return LBM_EINVAL;
  if (!g->bound) return LBM_ESTATE;
  DeviceScope dev(g->device);
  unsigned long long h[2] = {0ull, 0ull};
  CK(cudaMemcpyAsync(h, (const char*)g->d_status + NEWTON_COUNTER_OFFSET, sizeof(h), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  if (iterations) *iterations = (int64_t)h[0];
  if (solves) *solves = (int64_t)h[1];
  return LBM_OK;
}

const char* lbm_kernel_name(const lbm_grid* g) {
  if (!g) return "";
  if (g->matrix) return g->ks->matrix_name;
  return (g->pipe && g->hg.lv[0].n >= g->pipe_min_cells) ? g->ks->pipe_name : g->bricks ? g->ks->bricks_name : g->ks->name;
}

int lbm_get_macroscopic(lbm_grid* g, double* rho, double* ux, double* uy, double* T) {
  if (!g) return LBM_EINVAL;
  if (!g->bound || !g->inited) return LBM_ESTATE;
  DeviceScope dev(g->device);
  const size_t N = (size_t)g->n_total;
  double* d[4] = {g->d_scratch, g->d_scratch + N, g->d_scratch + 2 * N, g->d_scratch + 3 * N};
  if (g->matrix) {
    MatrixArgs ma = matrix_args(g, g->dl[0].cur);
    ma.o_rho = d[0]; ma.o_ux = d[1]; ma.o_uy = d[2]; ma.o_T = d[3];
    int rc = launch(g->ks->matrix_macro, g->dl[0].n, &ma, &g->mp, g->stream);
    if (rc) return rc;
  }
  int64_t base = 0;
  for (int l = 0; l <= g->depth && !g->matrix; ++l) {
    DevLevel& L = g->dl[l];
    MacroArgs a;
    a.n = (int)L.n; a.ps = L.ps; a.S = L.S[L.cur]; a.cells = nullptr;
    a.rho = d[0] + base; a.ux = d[1] + base; a.uy = d[2] + base; a.Tm = d[3] + base;
    int rc = launch(g->ks->macro, L.n, &a, &g->mp, g->stream);
    if (rc) return rc;
    base += L.n;
  }
  double* h[4] = {rho, ux, uy, T};
  for (int k = 0; k < 4; ++k)
    if (h[k]) CK(cudaMemcpyAsync(h[k], d[k], N * 8, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return LBM_OK;
}

int lbm_get_sensor(lbm_grid* g, double* eps) {
  if (!g || !eps) return LBM_EINVAL;
  if (!g->bound || !g->inited) return LBM_ESTATE;
  DeviceScope dev(g->device);
  const size_t N = (size_t)g->n_total;
  double* d = g->d_scratch;
  if (g->matrix) {
    MatrixArgs ma = matrix_args(g, g->dl[0].cur);
    ma.o_rho = d;
    int rc = launch(g->ks->matrix_sensor, g->dl[0].n, &ma, &g->mp, g->stream);
    if (rc) return rc;
  } else {
    int64_t base = 0;
    for (int l = 0; l <= g->depth; ++l) {
      DevLevel& L = g->dl[l];
      SensorArgs a;
      a.n = (int)L.n; a.ps = L.ps; a.S = L.S[L.cur]; a.eps = d + base;
      int rc = launch(g->ks->sensor_field, L.n, &a, &g->mp, g->stream);
      if (rc) return rc;
      base += L.n;
    }
  }
  CK(cudaMemcpyAsync(eps, d, N * 8, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return LBM_OK;
}

int lbm_get_macroscopic_at(lbm_grid* g, int l, int n, const int32_t* cells, double* rho, double* ux, double* uy, double* T) {
  if (!g || !cells || n < 0 || l < 0 || l > g->depth) return LBM_EINVAL;
  if (!g->bound || !g->inited) return LBM_ESTATE;
  if (n == 0) return LBM_OK;
  DeviceScope dev(g->device);
  DevLevel& L = g->dl[l];
  if ((size_t)n * 5 + 8 > g->scratch_doubles) return LBM_EINVAL;
  for (int k = 0; k < n; ++k)
    if (cells[k] < 0 || cells[k] >= L.n) return LBM_EINVAL;
  double* d[4] = {g->d_scratch, g->d_scratch + n, g->d_scratch + 2 * (size_t)n, g->d_scratch + 3 * (size_t)n};
  int* d_cells = (int*)(g->d_scratch + 4 * (size_t)n);
  CK(cudaMemcpyAsync(d_cells, cells, (size_t)n * 4, cudaMemcpyHostToDevice, g->stream));
  int rc;
  if (g->matrix) {
    MatrixArgs ma = matrix_args(g, L.cur);
    ma.n = n; ma.cells = d_cells; ma.o_rho = d[0]; ma.o_ux = d[1]; ma.o_uy = d[2]; ma.o_T = d[3];
    rc = launch(g->ks->matrix_macro, n, &ma, &g->mp, g->stream);
  } else {
    MacroArgs a;
    a.n = n; a.ps = L.ps; a.S = L.S[L.cur]; a.cells = d_cells;
    a.rho = d[0]; a.ux = d[1]; a.uy = d[2]; a.Tm = d[3];
    rc = launch(g->ks->macro, n, &a, &g->mp, g->stream);
  }
  if (rc) return rc;
  double* h[4] = {rho, ux, uy, T};
  for (int k = 0; k < 4; ++k)
    if (h[k]) CK(cudaMemcpyAsync(h[k], d[k], (size_t)n * 8, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return LBM_OK;
}

}  // extern "C"

// ---- lbm_get_macroscopic_at_static: the probe-cell read-out with its scratch in a file-scope device array instead of the
// caller's arena (for callers that hand the library no scratch area and may not allocate: include/lbm.h).  Layout of the
// array: [cells: MAX int32 | rho | ux | uy | T: MAX doubles each].  Every GPU that loads the library holds it until exit.
namespace {
constexpr int STATIC_PROBE_MAX = LBM_STATIC_PROBE_MAX;
constexpr size_t STATIC_PROBE_BYTES = (size_t)STATIC_PROBE_MAX * (4 + 4 * 8);
static __device__ __align__(256) unsigned char g_static_probe_scratch[STATIC_PROBE_BYTES];
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_probe_mutex;
void* g_static_probe_addr[STATIC_MAX_DEVICES] = {};     // device address of the array per device ordinal (0 = not asked yet)

// In host code the array's name is a host-side stand-in, not a device address: the address comes from cudaGetSymbolAddress,
// once per device, with that device current (the caller holds a DeviceScope).
int static_probe_scratch(int device, unsigned char** out) {
  if (device < 0 || device >= STATIC_MAX_DEVICES) return LBM_EINVAL;
  std::lock_guard<std::mutex> lock(g_static_probe_mutex);
  if (!g_static_probe_addr[device]) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_static_probe_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return LBM_ECUDA; }
    g_static_probe_addr[device] = ptr;
  }
  *out = (unsigned char*)g_static_probe_addr[device];
  return LBM_OK;
}
}  // namespace

extern "C" {

int lbm_get_macroscopic_at_static(lbm_grid* g, int l, int n, const int32_t* cells, double* rho, double* ux, double* uy, double* T) {
  if (!g || !cells || n < 0 || l < 0 || l > g->depth) return LBM_EINVAL;
  if (n > STATIC_PROBE_MAX) return LBM_ETOOLARGE;           // beyond the static scratch: use lbm_get_macroscopic_at
  if (!g->bound || !g->inited) return LBM_ESTATE;
  if (n == 0) return LBM_OK;
  DeviceScope dev(g->device);
  DevLevel& L = g->dl[l];
  for (int k = 0; k < n; ++k)
    if (cells[k] < 0 || cells[k] >= L.n) return LBM_EINVAL;
  unsigned char* base = nullptr;
  int rc = static_probe_scratch(g->device, &base);
  if (rc) return rc;
  int* d_cells = (int*)base;
  double* d0 = (double*)(base + (size_t)STATIC_PROBE_MAX * 4);
  double* d[4] = {d0, d0 + STATIC_PROBE_MAX, d0 + 2 * (size_t)STATIC_PROBE_MAX, d0 + 3 * (size_t)STATIC_PROBE_MAX};
  // the array keeps the previous call's contents; nothing in it has to start at zero: the n index slots are overwritten by
  // this copy and the 4 n output slots by the kernel before anything reads them, and only those are copied back
  CK(cudaMemcpyAsync(d_cells, cells, (size_t)n * 4, cudaMemcpyHostToDevice, g->stream));
  if (g->matrix) {
    MatrixArgs ma = matrix_args(g, L.cur);
    ma.n = n; ma.cells = d_cells; ma.o_rho = d[0]; ma.o_ux = d[1]; ma.o_uy = d[2]; ma.o_T = d[3];
    rc = launch(g->ks->matrix_macro, n, &ma, &g->mp, g->stream);
  } else {
    MacroArgs a;
    a.n = n; a.ps = L.ps; a.S = L.S[L.cur]; a.cells = d_cells;
    a.rho = d[0]; a.ux = d[1]; a.uy = d[2]; a.Tm = d[3];
    rc = launch(g->ks->macro, n, &a, &g->mp, g->stream);
  }
  if (rc) return rc;
  double* h[4] = {rho, ux, uy, T};
  for (int k = 0; k < 4; ++k)
    if (h[k]) CK(cudaMemcpyAsync(h[k], d[k], (size_t)n * 8, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return LBM_OK;
}

int lbm_get_populations(lbm_grid* g, int l, int which, double* out) {
  if (!g || !out || l < 0 || l > g->depth) return LBM_EINVAL;
  if (!g->bound) return LBM_ESTATE;
  int off, cnt;
  if (pop_range(g, which, &off, &cnt)) return LBM_EINVAL;
  DeviceScope dev(g->device);
  DevLevel& L = g->dl[l];
  if (L.n == 0) return LBM_OK;
  const long long tot = (long long)L.n * cnt;
  const unsigned grid = (unsigned)((tot + 255) / 256);
  if (g->matrix) {
    MatrixArgs ma = matrix_args(g, L.cur);
    ma.pops = g->d_scratch;
    int rc = launch(g->ks->matrix_export, L.n, &ma, &g->mp, g->stream);
    if (rc) return rc;
  } else if (g->esize == 8)
    export_kernel<double><<<grid, 256, 0, g->stream>>>((const double*)L.S[L.cur], L.ps, (int)L.n, off, cnt, g->d_scratch);
  else
    export_kernel<float><<<grid, 256, 0, g->stream>>>((const float*)L.S[L.cur], L.ps, (int)L.n, off, cnt, g->d_scratch);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(out, g->d_scratch, (size_t)tot * 8, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return LBM_OK;
}

int lbm_set_populations(lbm_grid* g, int l, int which, const double* in) {
  if (!g || !in || l < 0 || l > g->depth) return LBM_EINVAL;
  if (!g->bound) return LBM_ESTATE;
  int off, cnt;
  if (pop_range(g, which, &off, &cnt)) return LBM_EINVAL;
  DeviceScope dev(g->device);
  DevLevel& L = g->dl[l];
  if (L.n == 0) return LBM_OK;
  const long long tot = (long long)L.n * cnt;
  const unsigned grid = (unsigned)((tot + 255) / 256);
  CK(cudaMemcpyAsync(g->d_scratch, in, (size_t)tot * 8, cudaMemcpyHostToDevice, g->stream));
  if (g->matrix) {
    MatrixArgs ma = matrix_args(g, L.cur);
    ma.pops = g->d_scratch;
    int rc = launch(g->ks->matrix_import, L.n, &ma, &g->mp, g->stream);
    if (rc) return rc;
  } else if (g->esize == 8)
    import_kernel<double><<<grid, 256, 0, g->stream>>>((double*)L.S[L.cur], L.ps, (int)L.n, off, cnt, g->d_scratch);
  else
    import_kernel<float><<<grid, 256, 0, g->stream>>>((float*)L.S[L.cur], L.ps, (int)L.n, off, cnt, g->d_scratch);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(g->stream));
  g->inited = true;
  return LBM_OK;
}

}  // extern "C"
