/*
 * lbm.h -- C ABI of the B200-native quadtree lattice-Boltzmann hot path
 * (after Coreixas & Latt, arXiv 2504.04465; PAPER.md lines cited as P:<n>).
 *
 * The library runs, entirely in hand-written sm_100a CUDA kernels, the per-time-step fused
 * collide-and-stream update (Eq. 30-31) over a cell-centred, Morton-ordered quadtree
 * with int32 neighbour-list addressing (Sec. 4.3-4.4), Rohde-style coalescence /
 * uniform explosion (Eq. 4-7) and asynchronous time stepping (listing P:202-215).
 * The host only builds the mesh tables once.  There is no CPU fallback: every compute entry
 * point returns LBM_ECUDA when no device is usable.
 *
 * Conventions
 *  - Level 0 = finest, level `depth` = coarsest.  One coarse step = 2^depth fine steps.
 *  - A cell of level l at integer position (ix,iy) has its centre at ((ix+1/2)h,(iy+1/2)h), h=2^l.
 *  - Storage order of a level: in-box cells along the Z-curve with x in the even bits,
 *    then boundary cells by (iy,ix).  Storage index = rank in that order (int32).
 *  - Canonical direction order: index 0 = rest, then the groups of Table 4 in row order,
 *    inside a group counter-clockwise from +x.
 *  - State of a stored cell = POST-collision populations f*_i (Eq. 30), g*_i (Eq. 50) and the
 *    multipliers lambda (Eq. 39) that produced them.
 *  - All per-cell HOST arrays are flat over levels 0..depth in storage order (level l starts at
 *    sum_{m<l} N_m) and are owned by the caller.  Host I/O is always double; conversion to the
 *    grid's precision happens on the device.
 *  - Ownership: the handle and the host-side mesh tables belong to the library; DEVICE memory (one
 *    arena sized by lbm_grid_query) and the CUDA stream belong to the caller.
 *  - Every function returns 0 on success or a negative LBM_E* code.  No exceptions cross the ABI,
 *    no global state.  Functions taking a grid are not thread-safe on the same grid.
 */
#ifndef LBM_H
#define LBM_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LBM_MAX_LEVELS 24
#define LBM_QMAX 37
#define LBM_NLAMBDA 8
#define LBM_STATIC_PROBE_MAX 4096   /* probe cells per lbm_get_macroscopic_at_static call (144 KB of static device memory) */

/* collision models: BGK with polynomial equilibrium (Eq. 30, 34), recursive regularised (Eq. 33-38),
 * BGK with numerical equilibrium (Eq. 39-49) */
enum { LBM_BGK = 0, LBM_RR = 1, LBM_NUMEQ = 2 };
/* boundary kind per side; sides: 0 = x<0, 1 = x>=nx, 2 = y<0, 3 = y>=ny */
enum { LBM_BC_PERIODIC = 0, LBM_BC_WALL = 1, LBM_BC_MOVING_WALL = 2, LBM_BC_INFLOW_VBB = 3,
       LBM_BC_DIRICHLET_EQ = 4, LBM_BC_DIRICHLET_EQ_RHO_EXTRAP = 5, LBM_BC_NEUMANN = 6 };
/* cell types */
enum { LBM_FLUID = 0, LBM_FINE_GHOST = 1, LBM_COARSE_GHOST = 2, LBM_NEUMANN = 3, LBM_DIRICHLET = 4 };
/* negative link values in the neighbour list */
enum { LBM_LINK_NONE = -1, LBM_LINK_WALL = -2, LBM_LINK_VBB0 = -3 /* -3-side */ };
/* device addressing modes (lbm_config.addressing) */
enum { LBM_ADDR_AUTO = 0, LBM_ADDR_LIST = 1, LBM_ADDR_BRICKS = 2, LBM_ADDR_MATRIX = 3 };
/* software-pipelined sweep of the wide models (lbm_config.pipeline) */
enum { LBM_PIPE_AUTO = 0, LBM_PIPE_OFF = 1, LBM_PIPE_ALWAYS = 2 };
/* error codes */
enum { LBM_OK = 0, LBM_EINVAL = -1, LBM_ENOMEM = -2, LBM_EMESH = -3, LBM_ECUDA = -4,
       LBM_EUNSTABLE = -5 /* non-finite or non-positive density */,
       LBM_ENEWTON = -6 /* Newton-Raphson did not converge */,
       LBM_EUNSUPPORTED = -7 /* model combination has no compiled kernel */,
       LBM_ESTATE = -8 /* call order: not bound / not initialised */,
       LBM_ETOOLARGE = -9 /* request beyond a fixed capacity (lbm_get_macroscopic_at_static: LBM_STATIC_PROBE_MAX) */ };

typedef struct {
  int lattice;        /* 9, 13, 21, 37 (Table 4) */
  int precision;      /* 64 or 32: storage and arithmetic type of the populations */
  int collision;      /* LBM_BGK | LBM_RR | LBM_NUMEQ */
  int ddf;            /* 1: second distribution g, Eq. 50-51 */
  int sensor;         /* 1: kinetic shock sensor, Eq. 52-53 */
  int trace_eq;       /* RR only: trace of the 2nd-order non-equilibrium moments relaxed with tau=1 */
  int depth;          /* number of levels - 1 */
  int nx_coarse, ny_coarse;   /* box of the coarsest level, in coarsest cells */
  int newton_max_iter;        /* P:903; S14 */
  int bc[4];
  double tau0;        /* relaxation time of the finest level; tau_l = 1/2 + (tau0-1/2)/2^l (Eq. 3) */
  double T0;          /* reference temperature of numerical equilibria; polynomial models use c_s^2 */
  double gamma;       /* specific-heat ratio of the ddf model */
  double sensor_A;    /* Eq. 53 */
  double newton_tol;  /* sum_a |G_a| <= newton_tol rho; single precision: within 32 newton_tol at the iteration limit (S27) */
  double bc_rho[4], bc_ux[4], bc_uy[4], bc_T[4];   /* imposed states per side (walls: velocity only) */
  /* Pressure-relaxation sponge against acoustic reflections, Eq. 10-11 P:296-303 (reading S24 of DESIGN.md):
   * sigma(r) = 0 for r < r0, rises linearly to sigma_max at r1 and stays there, r = distance of the cell centre from
   * (x0, y0) in finest-level units; before each collision rho is relaxed to rho (1 - sigma) + sigma rho_inf at unchanged
   * velocity and non-equilibrium part.  sigma_max = 0: off.  Weakly compressible models only (LBM_EINVAL otherwise). */
  double sponge_x0, sponge_y0, sponge_r0, sponge_r1, sponge_sigma_max, sponge_rho_inf;
  /* Device-path options (they change how the kernels address memory and how launches are chained, never the result):
   * addressing: LBM_ADDR_AUTO = regular 8x8 bricks by tile arithmetic on levels of >= 2^18 stored cells and the neighbour
   * list elsewhere; LBM_ADDR_LIST = the list-addressed kernel of north_star on every level;
   * LBM_ADDR_BRICKS = bricks on every level that has some; LBM_ADDR_MATRIX = the "matrix-like" path of P:512-522 / P:744:
   * Cartesian-index addressing (no list, no type on the device) with AA-pattern in-place streaming, ONE population copy
   * (arena_bytes about halves), for single-level boxes (depth 0) without solids or sponge whose sides are periodic,
   * walls or moving walls, weakly compressible models only -- anything else: LBM_EINVAL.  Host tables and the order of
   * all host arrays stay the Z-curve storage order.  no_pdl = 1: plain stream order between level sweeps instead
   * of programmatic dependent launch edges.  pipeline: the wide models (second distribution and / or numerical equilibria)
   * run a software-pipelined persistent sweep (gathers of a thread's next cell in flight as cp.async while it computes the
   * current one): LBM_PIPE_AUTO = where it was measured faster (D2Q13 fp32 numerical equilibria), on levels
   * that give every resident thread at least two cells,
   * LBM_PIPE_OFF = never (one cell per thread everywhere), LBM_PIPE_ALWAYS = on every level.  pipe_max_ctas > 0 caps the
   * grid of that sweep (default 0: every resident CTA slot of the device), so that threads walk over more cells.
   * no_prefetch = 1: the one-cell-per-thread sweep of the wide models does not request the next wave's link rows and
   * population lines into the L2.  concurrent_levels = 1 (trees of >= 3 levels): in the graphs of
   * lbm_step the updates of levels >= 2 of a fine step run on a side branch beside the level-0 update of the next fine step
   * (the overlap proposed; U(0, k+1) depends on U(1, k) only), joined before the next update of level 1; programmatic
   * dependent launch is then off.  Measured +0.1 % on the six-level cylinder, hence off by default. */
  int addressing;
  int no_pdl;
  int pipeline;
  int pipe_max_ctas;
  int no_prefetch;
  int concurrent_levels;
} lbm_config;

typedef struct {
  int depth, Q, W;              /* W = lattice reach = ghost-band width in coarse cells */
  int npop;                     /* reals per cell: Q (+Q with g) (+8 with numerical equilibria) */
  int precision;
  int64_t n_cells[LBM_MAX_LEVELS];        /* stored cells per level, ghosts and boundary cells included */
  int64_t n_inbox[LBM_MAX_LEVELS];        /* of which inside the box (Morton-ordered part) */
  int64_t n_coarse_ghosts[LBM_MAX_LEVELS];/* coarse ghosts of interface (l, l-1); 0 for l = 0 */
  int64_t n_fine_ghosts[LBM_MAX_LEVELS];
  int64_t n_total;                        /* sum of n_cells */
  int64_t updates_per_coarse_step;        /* sum_l n_cells[l] * 2^(depth-l): actual cell updates */
  int64_t launches_per_coarse_step;       /* kernels enqueued per coarse step */
  size_t  arena_bytes;                    /* device memory the caller must provide to lbm_grid_bind */
  double  tau[LBM_MAX_LEVELS];
  int64_t n_bricks[LBM_MAX_LEVELS];       /* regular 8x8 bricks (64 cells each) addressed by tile arithmetic on the device */
  int64_t brick_min_level_cells;          /* levels with fewer stored cells go through the list (latency-bound) */
} lbm_grid_info;

typedef struct lbm_grid lbm_grid;   /* opaque */

/* Builds the quadtree levels, Morton order, neighbour lists, ghost lists and the level schedule on the
 * HOST (Sec. 4.3-4.4; rules: DESIGN.md Sec. 6).  No CUDA call is made.
 * Mesh = internal nodes + solid positions: split_xy / solid_xy are flat HOST (ix,iy) int32 pairs, the
 * cells of level l occupy pairs [off[l], off[l+1]) (off has depth+2 entries; level 0 has no split
 * cells); either pair of pointers may be NULL (= empty).  Returns LBM_EMESH if the mesh violates the
 * 2:1 / ghost-band rules, LBM_EUNSUPPORTED if the model combination has no compiled kernel. */
int lbm_grid_create(const lbm_config* cfg,
                    const int64_t* split_off, const int32_t* split_xy,
                    const int64_t* solid_off, const int32_t* solid_xy,
                    lbm_grid** out);
void lbm_destroy(lbm_grid* g);

int lbm_grid_query(const lbm_grid* g, lbm_grid_info* out);

/* Enumerates the model combinations this build has kernels for: fills lattice, precision, collision, ddf, sensor of *out
 * (everything else zero) for index = 0, 1, ... and returns LBM_EINVAL past the last one.  Any other combination makes
 * lbm_grid_create return LBM_EUNSUPPORTED.  HOST out.  No CUDA call. */
int lbm_supported_model(int index, lbm_config* out);

/* Bit-exact tables (HOST outputs, caller-owned, any may be NULL):
 *  cells:    ix, iy, type, aux per stored cell (aux: ghost-list index of a coarse ghost, source cell of a
 *            Neumann / Dirichlet cell, -1 otherwise)
 *  nbr:      n_cells*(Q-1) int32, row-major per cell: pull source of direction i (cell at x - xi_i) at
 *            [cell*(Q-1)+i-1], or a negative LBM_LINK_* value
 *  ghosts:   per coarse ghost of level l >= 1: its storage index, its 4 children on level l-1 in order
 *            a+2b (-1 absent), and the Q-bit mask of unknown directions
 *  schedule: canonical (pull) form of listing P:202-215: for fine step k = 1..2^depth the levels updated,
 *            ascending; returns the number of entries (writes at most cap). */
int lbm_get_cells(const lbm_grid* g, int level, int32_t* ix, int32_t* iy, int32_t* type, int32_t* aux);
int lbm_get_nbr(const lbm_grid* g, int level, int32_t* nbr);
int lbm_get_ghosts(const lbm_grid* g, int level, int32_t* coarse, int32_t* child, uint64_t* mask);
int lbm_get_schedule(const lbm_grid* g, int32_t* k_of, int32_t* level_of, int cap);
/* sponge coefficient sigma of every stored cell of one level (Eq. 11; HOST out, n_cells[level] doubles; zeros when off) */
int lbm_get_sponge(const lbm_grid* g, int level, double* sigma);
/* Compressed addressing of the device path: a "brick" is an aligned 8x8 tile of level-`level`
 * cells that are all stored FLUID cells (hence 64 consecutive storage indices) and whose
 * every neighbour-list entry equals  tiles9[9*b + k] + z  with (k, z) = (table[(i-1)*64 + m] >> 6, & 63) for the
 * cell at Z-position m and direction i: k = 3*ky + kx numbers the 3x3 tiles around the brick (k = 4: itself),
 * tiles9 holds the storage index of their first cell, z is the Z-position of the pull source in its tile.  The
 * builder verifies every brick against the list entry by entry; cells outside bricks use the list.
 * tiles9: HOST out, 9*n_bricks[level] int32; table: HOST out, (Q-1)*64 uint16; either may be NULL. */
int lbm_get_bricks(const lbm_grid* g, int level, int32_t* tiles9, uint16_t* table);

/* Attaches caller-owned DEVICE memory (>= arena_bytes, 256-byte aligned, on the CURRENT device of the calling thread)
 * and a CUDA stream of that device (cudaStream_t passed as void*; NULL = the library creates and owns a non-blocking
 * stream) and uploads the mesh tables.  The device is remembered: every later call on this grid selects it for its own
 * duration and restores the caller's current device before returning.  The CUDA graphs of the coarse step are captured on
 * first use by lbm_step.  The arena must stay valid until lbm_destroy.  On failure nothing stays attached. */
int lbm_grid_bind(lbm_grid* g, void* dev_arena, size_t nbytes, void* cuda_stream);

/* Sets every stored cell (ghosts included) to the equilibrium of the given macroscopic fields at its own
 * centre, then runs the iteration-0 coupling (coalesce unknown -> collide -> explode,
 * l = depth..1) without streaming (listing P:202-208).  rho, ux, uy, T: HOST arrays of n_total doubles
 * (T may be NULL = T0; ignored by athermal models).  Computed on the device.  Synchronises. */
int lbm_init_fields(lbm_grid* g, const double* rho, const double* ux, const double* uy, const double* T);

/* Enqueues n_coarse_steps coarse steps (each 2^depth fine steps of the schedule above) on the bound
 * stream and returns without synchronising. */
int lbm_step(lbm_grid* g, int n_coarse_steps);
/* Enqueues n FINE steps of the same schedule (fine step k updates level 0, then every level l with k = 0 mod 2^l,
 * ascending; listing P:202-215 in pull form) as plain kernel launches, continuing from wherever the previous call
 * stopped inside the coarse step.  For tests and for timing sub-steps; lbm_step returns LBM_ESTATE unless the
 * fine-step count since the last coarse-step boundary is a multiple of 2^depth.  lbm_init_fields resets the count. */
int lbm_step_fine(lbm_grid* g, int n_fine_steps);
/* Time-dependent parameters of the paper's start-up ramps: the viscosity ramp (nu lowered linearly from 100 nu to nu
 * over 20 convective times) is a sequence of lbm_set_relaxation calls (tau0 >= 1/2 of the finest level; tau_l follows Eq. 3),
 * the Mach ramp (the state imposed by the Dirichlet / velocity-bounce-back sides raised to its nominal value over one
 * convective time) a sequence of lbm_set_boundary_state calls (side 0..3; rho, u, T as in lbm_config).  Both take effect from
 * the next lbm_step / lbm_step_fine call; they synchronise the stream and drop the captured graphs, which are re-captured on
 * the next lbm_step (a few hundred microseconds: meant to be called once per coarse step, not per fine step). */
int lbm_set_relaxation(lbm_grid* g, double tau0);
int lbm_set_boundary_state(lbm_grid* g, int side, double rho, double ux, double uy, double T);
/* Mesh adaptation (Sec. 8.1).  `dst` is a grid over the same box with the same model
 * (lattice, precision, collision, ddf) and another tree, created with lbm_grid_create and bound to its own arena on the
 * same device; `src` is initialised and stands at a coarse-step boundary.  Every stored cell of dst (ghost and boundary
 * cells included) receives, on the device: the state of the cell src stores at the same level and place (copy); else the
 * state of the nearest stored ancestor (uniform explosion, Eq. 5, 7); else the mean over the children that have data, each
 * by copy or coalescence in turn (Eq. 4, 6: the area-weighted mean of the old cells it covers; children inside solids do
 * not exist); a Neumann cell follows its source cell.  Populations, g and the multipliers lambda alike.  The look-up runs on the
 * device too (binary search in the old tree's position keys, which the storage order keeps sorted); the host only uploads the keys
 * of the old and the positions of the new tree through the two scratch areas.  src's stream is synchronised first, the work runs on dst's stream, and
 * dst is initialised at fine step 0 afterwards (graphs are captured on its next lbm_step).  src stays valid.
 * LBM_EMESH: dst has a cell where src holds no data (the solids differ); LBM_EINVAL: models, boxes or devices differ, either
 * grid uses LBM_ADDR_MATRIX, or a cell is coarsened over more than three levels at once; LBM_ESTATE: not bound / not initialised / src inside a coarse step.  Synchronises. */
int lbm_transfer(lbm_grid* dst, lbm_grid* src);
/* Waits for the stream and returns the sticky device status: LBM_OK, LBM_EUNSTABLE or LBM_ENEWTON. */
int lbm_sync(lbm_grid* g);

/* rho, u (and T by Eq. 51) of every stored cell from its current populations; HOST outputs of
 * n_total doubles, any may be NULL.  Synchronises. */
int lbm_get_macroscopic(lbm_grid* g, double* rho, double* ux, double* uy, double* T);
/* The same for n probe cells of one level (storage indices in `cells`, HOST int32): time series without moving the whole
 * field (the steady-state, Strouhal and pressure-probe post-processing of Sec. 5 needs a few cells every few steps).
 * HOST outputs of n doubles, any may be NULL.  Synchronises.  LBM_EINVAL for an index outside the level. */
int lbm_get_macroscopic_at(lbm_grid* g, int level, int n, const int32_t* cells, double* rho, double* ux, double* uy, double* T);
/* lbm_get_macroscopic_at without any scratch from the caller and without any allocation: same arguments, same results
 * (the same kernel), but the staging area (the cell indices and the four output arrays on the device) is a file-scope
 * `static __device__` array of the library, LBM_STATIC_PROBE_MAX cells = 144 KB, which every GPU that loads the library
 * holds until the process exits.  For callers that may not allocate (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc) and do not want the library to touch the scratch part of their arena.  The call makes no
 * cudaMalloc / cudaFree and calls no allocating routine.  n > LBM_STATIC_PROBE_MAX: LBM_ETOOLARGE, nothing is done (use
 * lbm_get_macroscopic_at).  ALL grids of the process on one GPU share the one array and it keeps the last call's contents
 * (nothing in it needs to start at zero: every slot read is written first by the same call); two calls that overlap on the
 * GPU -- different grids on different streams, or two host threads -- race on it: serialise them.  Synchronises. */
int lbm_get_macroscopic_at_static(lbm_grid* g, int level, int n, const int32_t* cells, double* rho, double* ux, double* uy, double* T);
/* Refinement criterion of the paper's adaptive runs (the kinetic sensor, "the local departure to equilibrium"): eps of
 * Eq. 52, (1/V) sum_i |f_i - f_i^eq| / f_i^eq, of the CURRENT (post-collision) state of every stored cell, computed on the
 * device with the model's own equilibrium (numerical equilibria: from the stored multipliers); Eq. 30 scales f - f^eq by
 * (1 - 1/tau_eff), so this is |1 - 1/tau_eff| times the eps the last collision of the cell saw.  HOST output of n_total doubles
 * in storage order.  The caller thresholds it, builds the new tree and moves the state with lbm_transfer.  Synchronises. */
int lbm_get_sensor(lbm_grid* g, double* eps);
/* Current populations of one level as HOST doubles, row-major [cell][component];
 * which: 0 = f (Q), 1 = g (Q), 2 = lambda (8).  Synchronises. */
int lbm_get_populations(lbm_grid* g, int level, int which, double* out);
int lbm_set_populations(lbm_grid* g, int level, int which, const double* in);

/* Device-time of the work enqueued by the last lbm_step call, in milliseconds (CUDA events recorded on
 * the bound stream around it); synchronises.  Negative error code on failure. */
double lbm_last_step_ms(lbm_grid* g);
/* Newton statistics of the numerical-equilibrium models ("converges in just one iteration on average"):
 * Newton steps taken (the unconditional polish step of reading S14 included) and equilibrium solves performed on the device
 * since lbm_grid_bind (initialisation, iteration-0 coupling, every colliding or Dirichlet cell of every sweep), counted by
 * the kernels themselves.  HOST outputs, either may be NULL; zeros for polynomial models.  Synchronises. */
int lbm_newton_iterations(lbm_grid* g, int64_t* iterations, int64_t* solves);
/* Name of the compiled sweep kernel this grid dispatches to (static string), for profiles; says whether the
 * compressed addressing of regular bricks is in use (lbm_config.addressing). */
const char* lbm_kernel_name(const lbm_grid* g);


/* Measured FMA peak of the current device's plain fp64 (precision 64) or fp32 (32) pipe, in TFLOP/s (2 flop per
 * FMA): 8 independent dependent-FMA chains per thread, every SM filled to its thread limit, launches repeated for
 * about `seconds` of device time, best launch reported.  This is the denominator of the "alu" rooflines of the
 * D2Q37 and numerical-equilibrium paths (north_star: "FP64/FP32 pipe utilisation against peak").
 * tflops: HOST out.  lanes_mhz_per_sm (HOST out, may be NULL) = FMA/s per SM / 1e6 (= lanes x clock in MHz).
 * Uses the current device and the legacy default stream; allocates and frees one word.  LBM_ECUDA without a device. */
int lbm_measure_fma_peak(int precision, double seconds, double* tflops, double* lanes_mhz_per_sm);

#ifdef __cplusplus
}
#endif
#endif
