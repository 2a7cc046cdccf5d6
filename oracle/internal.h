/* internal.h -- CPU ORACLE (test infrastructure): structures shared by grid.c and sim.c. */
#ifndef ORACLE_INTERNAL_H
#define ORACLE_INTERNAL_H
#include "oracle.h"

typedef struct phys_t phys_t;   /* opaque here; defined in physics.c */
phys_t* orc_phys_new(const orc_config* cfg, int* rc);
int orc_phys_Q(const phys_t* P);
int orc_phys_W(const phys_t* P);
int orc_phys_cx(const phys_t* P, int i);
int orc_phys_cy(const phys_t* P, int i);
int orc_phys_opp(const phys_t* P, int i);
double orc_phys_w(const phys_t* P, int i);
double orc_phys_cs2(const phys_t* P);
double orc_phys_T0(const phys_t* P);
void orc_phys_moments(const phys_t* P, const double* f, const double* g, double* rho, double* ux, double* uy, double* T);
int orc_phys_equilibrium(const phys_t* P, double rho, double ux, double uy, double T, double* lam, double* feq, double* geq);
int orc_phys_collide(const phys_t* P, double tau, const double* f, const double* g, double* lam, double* fout, double* gout);

typedef struct {
  int64_t n;            /* stored cells of this level (in-box Morton-ordered, then boundary cells) */
  int64_t n_inbox;
  int32_t *ix, *iy, *type, *aux;
  int32_t* nbr;         /* n*(Q-1): pull source of direction i at [cell*(Q-1)+i-1] */
  int64_t ng;           /* coarse ghosts on this level (interface with level-1) */
  int32_t* g_coarse;    /* storage index of the coarse ghost */
  int32_t* g_child;     /* 4 per ghost: storage index on level-1 of child a+2b, -1 if absent */
  uint64_t* g_mask;     /* bit i set: direction i unknown (coalesced) */
  double tau;
  double* sigma;        /* sponge coefficient per stored cell (Eq. 11), NULL when the sponge is off */
  double* S[2];         /* populations, AoS [cell][npop]: f(Q) | g(Q) | lambda(8) */
  int cur;              /* which of S[] is current */
} orc_level;

struct orc_grid {
  orc_config cfg;
  phys_t* phys;
  int Q, W, npop;
  int depth;
  orc_level* lv;        /* depth+1 */
  int64_t k;            /* fine-step counter */
  int64_t newton_its;
  int64_t cell_updates;
  int status;           /* sticky error (ORC_EUNSTABLE / ORC_ENEWTON) */
};

int orc_build_levels(orc_grid* g, const int64_t* split_off, const int32_t* split_xy,
                     const int64_t* solid_off, const int32_t* solid_xy);

#endif
