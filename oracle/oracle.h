/*
 * oracle.h -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-threaded, double-precision restatement of the hot path of
 * Coreixas & Latt, "Compressible lattice Boltzmann methods on non-uniform grids"
 * (arXiv 2504.04465; PAPER.md, cited below as P:<line>).  It follows the paper's
 * algorithm step by step (DESIGN.md lists every reading taken where the paper is
 * silent).  It shares no code, header, table or helper with the CUDA path under
 * paper_2504_04465_b200/csrc; only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.
 *
 * State convention: every stored cell holds the
 * POST-collision populations f*_i(x,t) of Eq. (30), i.e. the paper's state
 * after collision and before the streaming of Eq. (31); one update of a cell
 * gathers f*_i(x-xi_i,t) (pull form of Eq. 31), then collides.
 *
 * Parity status of each part is listed in DESIGN.md ("Pins"); long-run fields of the
 * 2-D Riemann / NACA workloads are "parity unpinned" beyond GPU-vs-oracle.
 */
#ifndef ORACLE_H
#define ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_QMAX 37
#define ORC_NLAMBDA 8

/* collision models */
enum { ORC_BGK = 0, ORC_RR = 1, ORC_NUMEQ = 2 };
/* boundary kinds per side; sides: 0 = x<0 (left), 1 = x>=nx (right), 2 = y<0 (bottom), 3 = y>=ny (top) */
enum { ORC_BC_PERIODIC = 0, ORC_BC_WALL = 1, ORC_BC_MOVING_WALL = 2, ORC_BC_INFLOW_VBB = 3,
       ORC_BC_DIRICHLET_EQ = 4, ORC_BC_DIRICHLET_EQ_RHO_EXTRAP = 5, ORC_BC_NEUMANN = 6 };
/* cell types */
enum { ORC_FLUID = 0, ORC_FINE_GHOST = 1, ORC_COARSE_GHOST = 2, ORC_NEUMANN = 3, ORC_DIRICHLET = 4 };
/* link sentinels in the neighbour list (negative) */
enum { ORC_LINK_NONE = -1, ORC_LINK_WALL = -2, ORC_LINK_VBB0 = -3 /* -3-side */ };
/* error codes */
enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -2, ORC_EMESH = -3, ORC_EUNSTABLE = -5, ORC_ENEWTON = -6 };

typedef struct {
  int lattice;      /* 9, 13, 21, 37 (Table 4) */
  int collision;    /* ORC_BGK (polynomial eq.), ORC_RR (Eq. 33-38), ORC_NUMEQ (Eq. 39-49, BGK relaxation) */
  int ddf;          /* second distribution g, Eq. 50-51 */
  int sensor;       /* Eq. 52-53 */
  int trace_eq;     /* RR only: trace of 2nd-order neq moments relaxed with tau=1 */
  int depth;        /* number of levels - 1; level 0 = finest */
  int nx_coarse, ny_coarse;
  int newton_max_iter;
  int bc[4];
  double tau0;      /* relaxation time of the finest level, Eq. 3 */
  double T0;        /* reference temperature; ignored (=c_s^2) for polynomial equilibria */
  double gamma;     /* specific-heat ratio for the ddf model */
  double sensor_A;  /* Eq. 53 */
  double newton_tol;/* P:934 */
  double bc_rho[4], bc_ux[4], bc_uy[4], bc_T[4];
  /* pressure-relaxation sponge, Eq. 10-11 P:296-303 (reading S24 of DESIGN.md): sigma(r) = 0 for r < r0, rises linearly to
   * sigma_max at r1 and stays there, r = distance of the cell centre from (x0, y0) in finest-level units; before each
   * collision rho is relaxed to rho(1-sigma) + sigma rho_inf.  sigma_max = 0: off.  Weakly compressible models only. */
  double sponge_x0, sponge_y0, sponge_r0, sponge_r1, sponge_sigma_max, sponge_rho_inf;
} orc_config;

typedef struct orc_grid orc_grid;

/* Mesh description = the quadtree's internal nodes + solid positions, per level.
 * split_xy / solid_xy are flat (ix,iy) int32 pairs; cells of level l occupy pairs
 * [off[l], off[l+1]) (off has depth+2 entries; level 0 has no split cells). */
int  orc_grid_create(const orc_config* cfg,
                     const int64_t* split_off, const int32_t* split_xy,
                     const int64_t* solid_off, const int32_t* solid_xy,
                     orc_grid** out);
void orc_grid_destroy(orc_grid* g);

int     orc_depth(const orc_grid* g);
int64_t orc_num_cells(const orc_grid* g, int level);
int64_t orc_num_ghosts(const orc_grid* g, int level);   /* coarse ghosts of interface (level, level-1) */
double  orc_tau(const orc_grid* g, int level);
/* start-up ramps (P:333 viscosity ramp, P:424 Mach ramp): new tau_0 (tau_l by Eq. 3) / new imposed state of one side,
 * effective from the next update */
int  orc_get_sponge(const orc_grid* g, int level, double* sigma /* one per stored cell */);
int  orc_set_tau0(orc_grid* g, double tau0);
int  orc_set_bc_state(orc_grid* g, int side, double rho, double ux, double uy, double T);
/* storage-order tables of one level (caller-owned outputs, any may be NULL) */
int  orc_get_cells(const orc_grid* g, int level, int32_t* ix, int32_t* iy, int32_t* type, int32_t* aux);
int  orc_get_nbr(const orc_grid* g, int level, int32_t* nbr /* N*(Q-1), AoS, pull sources */);
int  orc_get_ghosts(const orc_grid* g, int level, int32_t* coarse, int32_t* child /* 4 per ghost */, uint64_t* mask);
/* schedule of one coarse step: for k=1..2^depth, levels updated (ascending); returns count written */
int  orc_get_schedule(const orc_grid* g, int32_t* k_of, int32_t* level_of, int cap);

/* fields are flat over levels 0..depth in storage order (level l starts at sum_{m<l} N_m) */
int  orc_init_fields(orc_grid* g, const double* rho, const double* ux, const double* uy, const double* T);
int  orc_step(orc_grid* g, int n_coarse_steps);
int  orc_step_fine(orc_grid* g, int n_fine_steps);     /* advances k by n fine steps (for 1000-fine-step parity) */
int  orc_get_macroscopic(const orc_grid* g, double* rho, double* ux, double* uy, double* T);
/* eps of Eq. 52 of the current state of every stored cell (flat over levels): the refinement criterion of P:717 */
int  orc_get_sensor(orc_grid* g, double* eps);
/* which: 0 = f (Q per cell), 1 = g (Q per cell), 2 = lambda (8 per cell); AoS [cell][component] */
int  orc_get_populations(const orc_grid* g, int level, int which, double* out);
int  orc_set_populations(orc_grid* g, int level, int which, const double* in);
int  orc_set_fine_step(orc_grid* g, int64_t k);         /* fine steps taken so far (schedule position), with an imported state */
/* Mesh adaptation (Sec. 8.1): moves the state of `src` (at a coarse-step boundary) onto `dst`, another tree over the
 * same box with the same model: copy where the old tree stores the cell, uniform explosion from the nearest stored ancestor,
 * else coalescence of the children (amr.c).  dst is then initialised at fine step 0.  ORC_EMESH if dst has a cell the old
 * tree holds no data for. */
int  orc_transfer(orc_grid* dst, const orc_grid* src);
int64_t orc_newton_iterations(const orc_grid* g);      /* total Newton iterations since create */
int64_t orc_cell_updates(const orc_grid* g);           /* total cell updates since create */

/* ---- cell-local pieces, exported so that the pins can test them in isolation ---- */
int  orc_lattice(int Q, int* cx, int* cy, double* w, int* opp, double* cs2, int* reach);
/* polynomial equilibrium Eq. 34 (thermal=0: athermal moments Eq. 36; thermal=1: T-dependent moments) */
int  orc_feq_poly(int Q, double rho, double ux, double uy, double T, int thermal, double* feq);
/* numerical equilibrium Eq. 39-49; lambda in/out; returns iterations (<0 on failure) */
int  orc_feq_numerical(int Q, double rho, double ux, double uy, double T, double tol, int max_iter,
                       double* lambda, double* feq);
/* one collision of a single cell (f,g in: pre-collision; out: post-collision); returns iterations */
int  orc_collide_cell(const orc_config* cfg, double tau, const double* f, const double* g,
                      double* lambda, double* fout, double* gout);

#ifdef __cplusplus
}
#endif
#endif
