/*
 * sim.c -- CPU ORACLE (test infrastructure): the level update (gather, coalesce, collide,
 * explode), the asynchronous schedule (listing P:202-215 in pull form), initialisation
 * and the C entry points declared in oracle.h.
 * Single thread, fp64, one cell after the other in storage order.
 */
#include "internal.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

static int dirichlet_side(const orc_grid* g, int l, int64_t c)
{
  const orc_level* L = &g->lv[l];
  const int nx = g->cfg.nx_coarse << (g->depth - l), ny = g->cfg.ny_coarse << (g->depth - l);
  const int ox = L->ix[c] < 0 ? 0 : (L->ix[c] >= nx ? 1 : -1);
  const int oy = L->iy[c] < 0 ? 2 : (L->iy[c] >= ny ? 3 : -1);
  return oy >= 0 ? oy : ox;
}

/* coalescence Eq. 4 / Eq. 6: mean over the children that exist of component p of their current state */
static double coalesce(const orc_grid* g, int l, int64_t ghost, int p)
{
  const orc_level* L = &g->lv[l];
  const orc_level* F = &g->lv[l - 1];
  const double* Sf = F->S[F->cur];
  double s = 0.0; int nf = 0;
  for (int ch = 0; ch < 4; ++ch) {
    const int32_t c = L->g_child[4 * ghost + ch];
    if (c < 0) continue;
    s += Sf[(int64_t)c * g->npop + p];
    ++nf;
  }
  return s / (double)nf;
}

/* uniform explosion Eq. 5 / Eq. 7: every child receives the coarse post-collision state */
static void explode(orc_grid* g, int l, int64_t ghost, const double* Sc)
{
  orc_level* L = &g->lv[l];
  orc_level* F = &g->lv[l - 1];
  double* Sf = F->S[F->cur];
  for (int ch = 0; ch < 4; ++ch) {
    const int32_t c = L->g_child[4 * ghost + ch];
    if (c < 0) continue;
    for (int p = 0; p < g->npop; ++p) Sf[(int64_t)c * g->npop + p] = Sc[p];
  }
}

static void check_state(orc_grid* g, const double* out, int it)
{
  double r = 0.0;
  for (int i = 0; i < g->Q; ++i) r += out[i];
  if (!(r > 0.0) || !isfinite(r)) g->status = ORC_EUNSTABLE;
  if (it < 0 && g->status == ORC_OK) g->status = ORC_ENEWTON;
  if (it != 0) g->newton_its += (it < 0 ? -it - 1 : it);
}

/* one update of level l: old buffer -> new buffer, coupling with level l-1 fused in (reading S15) */
static void update_level(orc_grid* g, int l)
{
  orc_level* L = &g->lv[l];
  const int Q = g->Q, np = g->npop, ddf = g->cfg.ddf, numeq = (g->cfg.collision == ORC_NUMEQ);
  const double* So = L->S[L->cur];
  double* Sn = L->S[1 - L->cur];
  const double cs2 = orc_phys_cs2(g->phys);
  double f[ORC_QMAX], gg[ORC_QMAX], lam[ORC_NLAMBDA], fo[ORC_QMAX], go[ORC_QMAX];

  for (int64_t c = 0; c < L->n; ++c) {
    const int type = L->type[c];
    double* out = Sn + c * np;
    if (type == ORC_DIRICHLET) {
      /* equilibrium Dirichlet cell: imposed state, rho optionally taken from the nearest interior cell */
      const int side = dirichlet_side(g, l, c);
      double rho = g->cfg.bc_rho[side];
      if (g->cfg.bc[side] == ORC_BC_DIRICHLET_EQ_RHO_EXTRAP) {
        const double* s = So + (int64_t)L->aux[c] * np;
        rho = 0.0;
        for (int i = 0; i < Q; ++i) rho += s[i];
      }
      const double T = (numeq || ddf) ? g->cfg.bc_T[side] : orc_phys_T0(g->phys);
      for (int a = 0; a < ORC_NLAMBDA; ++a) lam[a] = numeq ? So[c * np + (ddf ? 2 : 1) * Q + a] : 0.0;
      int it = orc_phys_equilibrium(g->phys, rho, g->cfg.bc_ux[side], g->cfg.bc_uy[side], T, lam, fo, go);
      for (int i = 0; i < Q; ++i) out[i] = fo[i];
      if (ddf) for (int i = 0; i < Q; ++i) out[Q + i] = go[i];
      if (numeq) for (int a = 0; a < ORC_NLAMBDA; ++a) out[(ddf ? 2 : 1) * Q + a] = lam[a];
      check_state(g, out, it);
      g->cell_updates++;
      continue;
    }
    /* NEUMANN replicates the update of its source cell (reading S13) */
    const int64_t self = (type == ORC_NEUMANN) ? L->aux[c] : c;
    const double* own = So + self * np;
    const int32_t* row = L->nbr + c * (Q - 1);
    /* step 1: gather (pull form of Eq. 31), boundary links */
    double rho_w = 0.0; int have_rho_w = 0;
    for (int i = 0; i < Q; ++i) {
      const int32_t n = (i == 0) ? (int32_t)self : row[i - 1];
      if (n >= 0) {
        f[i] = So[(int64_t)n * np + i];
        if (ddf) gg[i] = So[(int64_t)n * np + Q + i];
      } else if (n == ORC_LINK_WALL) {
        const int o = orc_phys_opp(g->phys, i);
        f[i] = own[o];
        if (ddf) gg[i] = own[Q + o];
      } else if (n <= ORC_LINK_VBB0) {
        /* velocity bounce-back (Ladd): f_i = f*_opp(i)(x) + 2 w_i rho_w (xi_i . u_w)/c_s^2, rho_w local (S11) */
        const int side = ORC_LINK_VBB0 - n;
        const int o = orc_phys_opp(g->phys, i);
        if (!have_rho_w) { for (int j = 0; j < Q; ++j) rho_w += own[j]; have_rho_w = 1; }
        const double xu = orc_phys_cx(g->phys, i) * g->cfg.bc_ux[side] + orc_phys_cy(g->phys, i) * g->cfg.bc_uy[side];
        f[i] = own[o] + 2.0 * orc_phys_w(g->phys, i) * rho_w * xu / cs2;
        if (ddf) gg[i] = own[Q + o];
      } else { /* ORC_LINK_NONE */
        if (type == ORC_COARSE_GHOST) {
          f[i] = coalesce(g, l, L->aux[c], i);                    /* Eq. 4 on unknown directions only */
          if (ddf) gg[i] = coalesce(g, l, L->aux[c], Q + i);
        } else {                                                  /* fine ghost without a source: keeps its value (S6) */
          f[i] = own[i];
          if (ddf) gg[i] = own[Q + i];
        }
      }
    }
    if (type == ORC_FINE_GHOST) {
      /* fine ghost cells stream without colliding */
      for (int i = 0; i < Q; ++i) out[i] = f[i];
      if (ddf) for (int i = 0; i < Q; ++i) out[Q + i] = gg[i];
      if (numeq) for (int a = 0; a < ORC_NLAMBDA; ++a) out[(ddf ? 2 : 1) * Q + a] = own[(ddf ? 2 : 1) * Q + a];
      g->cell_updates++;
      continue;
    }
    if (numeq) {
      const int off = (ddf ? 2 : 1) * Q;
      for (int a = 0; a < ORC_NLAMBDA; ++a)
        lam[a] = (type == ORC_COARSE_GHOST) ? coalesce(g, l, L->aux[c], off + a) /* Eq. 6 */ : own[off + a];
    }
    /* pressure relaxation (Eq. 10, "applied before the collision step"; reading S24): rho -> rho' = rho (1 - sigma) +
       sigma rho_inf at unchanged velocity and unchanged non-equilibrium part, i.e. f_i += (rho'/rho - 1) f_i^eq(rho, u)
       (the polynomial equilibrium is linear in rho); a Neumann cell follows its source cell (S13) */
    if (L->sigma && L->sigma[self] > 0.0) {
      const double sg = L->sigma[self];
      double rho = 0.0, jx = 0.0, jy = 0.0, dummy[ORC_NLAMBDA] = {0};
      for (int i = 0; i < Q; ++i) { rho += f[i]; jx += orc_phys_cx(g->phys, i) * f[i]; jy += orc_phys_cy(g->phys, i) * f[i]; }
      orc_phys_equilibrium(g->phys, rho, jx / rho, jy / rho, orc_phys_T0(g->phys), dummy, fo, go);
      const double rho_new = rho * (1.0 - sg) + sg * g->cfg.sponge_rho_inf;
      for (int i = 0; i < Q; ++i) f[i] += (rho_new / rho - 1.0) * fo[i];
    }
    /* steps 2-5: moments, equilibrium, sensor, relaxation */
    int it = orc_phys_collide(g->phys, L->tau, f, gg, lam, fo, go);
    for (int i = 0; i < Q; ++i) out[i] = fo[i];
    if (ddf) for (int i = 0; i < Q; ++i) out[Q + i] = go[i];
    if (numeq) for (int a = 0; a < ORC_NLAMBDA; ++a) out[(ddf ? 2 : 1) * Q + a] = lam[a];
    check_state(g, out, it);
    if (type == ORC_COARSE_GHOST) explode(g, l, L->aux[c], out);  /* Eq. 5, 7 */
    g->cell_updates++;
  }
  L->cur = 1 - L->cur;
}

/* one fine step in canonical (pull) form: level 0, then every level l with k = 0 mod 2^l, ascending */
static void fine_step(orc_grid* g)
{
  g->k++;
  update_level(g, 0);
  for (int l = 1; l <= g->depth; ++l) {
    if (g->k % ((int64_t)1 << l) != 0) break;
    update_level(g, l);
  }
}

int orc_step_fine(orc_grid* g, int n)
{
  for (int s = 0; s < n; ++s) fine_step(g);
  return g->status;
}

int orc_step(orc_grid* g, int n_coarse_steps)
{
  const int64_t per = (int64_t)1 << g->depth;
  for (int s = 0; s < n_coarse_steps; ++s)
    for (int64_t k = 0; k < per; ++k) fine_step(g);
  return g->status;
}

int orc_get_schedule(const orc_grid* g, int32_t* k_of, int32_t* level_of, int cap)
{
  int n = 0;
  const int64_t per = (int64_t)1 << g->depth;
  for (int64_t k = 1; k <= per; ++k)
    for (int l = 0; l <= g->depth; ++l) {
      if (l > 0 && k % ((int64_t)1 << l) != 0) break;
      if (n < cap) { if (k_of) k_of[n] = (int32_t)k; if (level_of) level_of[n] = l; }
      ++n;
    }
  return n;
}

/* ------------------------------------------------------------------ set-up */

int orc_grid_create(const orc_config* cfg, const int64_t* split_off, const int32_t* split_xy,
                    const int64_t* solid_off, const int32_t* solid_xy, orc_grid** out)
{
  if (!cfg || !out) return ORC_EINVAL;
  int rc = ORC_OK;
  orc_grid* g = (orc_grid*)calloc(1, sizeof(orc_grid));
  if (!g) return ORC_ENOMEM;
  g->cfg = *cfg;
  g->phys = orc_phys_new(cfg, &rc);
  if (!g->phys) { free(g); return rc; }
  g->Q = orc_phys_Q(g->phys); g->W = orc_phys_W(g->phys);
  g->depth = cfg->depth;
  g->npop = g->Q * (cfg->ddf ? 2 : 1) + (cfg->collision == ORC_NUMEQ ? ORC_NLAMBDA : 0);
  /* velocity bounce-back is defined for the weakly compressible models only */
  for (int s = 0; s < 4; ++s)
    if ((cfg->bc[s] == ORC_BC_MOVING_WALL || cfg->bc[s] == ORC_BC_INFLOW_VBB) && (cfg->ddf || cfg->collision == ORC_NUMEQ)) rc = ORC_EINVAL;
  if (!(cfg->tau0 >= 0.5)) rc = ORC_EINVAL;
  /* the sponge relaxes rho = p / T0: weakly compressible models only */
  if (cfg->sponge_sigma_max != 0.0 && (cfg->ddf || cfg->collision == ORC_NUMEQ || !(cfg->sponge_sigma_max > 0.0) ||
                                       !(cfg->sponge_sigma_max <= 1.0) || !(cfg->sponge_r1 > cfg->sponge_r0) || !(cfg->sponge_r0 >= 0.0)))
    rc = ORC_EINVAL;
  g->lv = (orc_level*)calloc((size_t)cfg->depth + 1, sizeof(orc_level));
  if (!g->lv) rc = ORC_ENOMEM;
  if (!rc) rc = orc_build_levels(g, split_off, split_xy, solid_off, solid_xy);
  for (int l = 0; l <= g->depth && !rc; ++l) {
    orc_level* L = &g->lv[l];
    /* Eq. 3 (reading S3): tau_l - 1/2 = (tau_0 - 1/2) / 2^l */
    L->tau = 0.5 + (cfg->tau0 - 0.5) / (double)((int64_t)1 << l);
    for (int b = 0; b < 2; ++b) {
      L->S[b] = (double*)calloc((size_t)(L->n * g->npop + 1), sizeof(double));
      if (!L->S[b]) rc = ORC_ENOMEM;
    }
    if (cfg->sponge_sigma_max > 0.0 && !rc) {
      /* Eq. 11: linear ramp of sigma between r0 and r1 around (x0, y0), cell centres ((ix+1/2)h, (iy+1/2)h), h = 2^l */
      L->sigma = (double*)calloc((size_t)L->n + 1, sizeof(double));
      if (!L->sigma) { rc = ORC_ENOMEM; break; }
      const double h = (double)((int64_t)1 << l);
      for (int64_t c = 0; c < L->n; ++c) {
        const double dx = (L->ix[c] + 0.5) * h - cfg->sponge_x0, dy = (L->iy[c] + 0.5) * h - cfg->sponge_y0;
        const double r = sqrt(dx * dx + dy * dy);
        double sg = 0.0;
        if (r >= cfg->sponge_r1) sg = cfg->sponge_sigma_max;
        else if (r >= cfg->sponge_r0) sg = cfg->sponge_sigma_max * (r - cfg->sponge_r0) / (cfg->sponge_r1 - cfg->sponge_r0);
        L->sigma[c] = sg;
      }
    }
  }
  if (rc) { orc_grid_destroy(g); return rc; }
  *out = g;
  return ORC_OK;
}

void orc_grid_destroy(orc_grid* g)
{
  if (!g) return;
  if (g->lv)
    for (int l = 0; l <= g->depth; ++l) {
      orc_level* L = &g->lv[l];
      free(L->ix); free(L->iy); free(L->type); free(L->aux); free(L->nbr);
      free(L->g_coarse); free(L->g_child); free(L->g_mask); free(L->S[0]); free(L->S[1]); free(L->sigma);
    }
  free(g->lv);
  free(g->phys);
  free(g);
}

int orc_depth(const orc_grid* g) { return g->depth; }
int64_t orc_num_cells(const orc_grid* g, int l) { return (l < 0 || l > g->depth) ? -1 : g->lv[l].n; }
int64_t orc_num_ghosts(const orc_grid* g, int l) { return (l < 1 || l > g->depth) ? 0 : g->lv[l].ng; }
double orc_tau(const orc_grid* g, int l) { return g->lv[l].tau; }

/* Time-dependent parameters of the start-up ramps (viscosity ramp P:333: nu decreased linearly from 100 nu to nu; Mach
 * ramp P:424: the state imposed by the Dirichlet sides raised to its nominal value): they act from the next update on.
 * tau_l follows Eq. 3 (reading S3) from the new tau_0. */
int orc_get_sponge(const orc_grid* g, int l, double* sigma) {
  if (!g || !sigma || l < 0 || l > g->depth) return ORC_EINVAL;
  for (int64_t c = 0; c < g->lv[l].n; ++c) sigma[c] = g->lv[l].sigma ? g->lv[l].sigma[c] : 0.0;
  return ORC_OK;
}

int orc_set_tau0(orc_grid* g, double tau0) {
  if (!g || !(tau0 >= 0.5)) return ORC_EINVAL;
  g->cfg.tau0 = tau0;
  for (int l = 0; l <= g->depth; ++l) g->lv[l].tau = 0.5 + (tau0 - 0.5) / (double)((int64_t)1 << l);
  return ORC_OK;
}

int orc_set_bc_state(orc_grid* g, int side, double rho, double ux, double uy, double T) {
  if (!g || side < 0 || side > 3) return ORC_EINVAL;
  g->cfg.bc_rho[side] = rho; g->cfg.bc_ux[side] = ux; g->cfg.bc_uy[side] = uy; g->cfg.bc_T[side] = T;
  return ORC_OK;
}
int64_t orc_newton_iterations(const orc_grid* g) { return g->newton_its; }
int64_t orc_cell_updates(const orc_grid* g) { return g->cell_updates; }

int orc_get_cells(const orc_grid* g, int l, int32_t* ix, int32_t* iy, int32_t* type, int32_t* aux)
{
  if (l < 0 || l > g->depth) return ORC_EINVAL;
  const orc_level* L = &g->lv[l];
  for (int64_t c = 0; c < L->n; ++c) {
    if (ix) ix[c] = L->ix[c];
    if (iy) iy[c] = L->iy[c];
    if (type) type[c] = L->type[c];
    if (aux) aux[c] = L->aux[c];
  }
  return ORC_OK;
}

int orc_get_nbr(const orc_grid* g, int l, int32_t* nbr)
{
  if (l < 0 || l > g->depth) return ORC_EINVAL;
  memcpy(nbr, g->lv[l].nbr, sizeof(int32_t) * (size_t)(g->lv[l].n * (g->Q - 1)));
  return ORC_OK;
}

int orc_get_ghosts(const orc_grid* g, int l, int32_t* coarse, int32_t* child, uint64_t* mask)
{
  if (l < 1 || l > g->depth) return ORC_EINVAL;
  const orc_level* L = &g->lv[l];
  if (coarse) memcpy(coarse, L->g_coarse, sizeof(int32_t) * (size_t)L->ng);
  if (child) memcpy(child, L->g_child, sizeof(int32_t) * (size_t)(4 * L->ng));
  if (mask) memcpy(mask, L->g_mask, sizeof(uint64_t) * (size_t)L->ng);
  return ORC_OK;
}

/* populations at the equilibrium of the given macroscopic fields at every stored cell,
 * then the coupling of iteration 0 without streaming (listing P:202-208): coalesce the unknown
 * directions of every coarse ghost, collide it, explode to its children. */
int orc_init_fields(orc_grid* g, const double* rho, const double* ux, const double* uy, const double* T)
{
  const int Q = g->Q, np = g->npop, ddf = g->cfg.ddf, numeq = (g->cfg.collision == ORC_NUMEQ);
  const int loff = (ddf ? 2 : 1) * Q;
  double feq[ORC_QMAX], geq[ORC_QMAX], lam[ORC_NLAMBDA];
  int64_t base = 0;
  g->k = 0; g->status = ORC_OK;
  for (int l = 0; l <= g->depth; ++l) {
    orc_level* L = &g->lv[l];
    L->cur = 0;
    for (int64_t c = 0; c < L->n; ++c) {
      const double r = rho[base + c], vx = ux[base + c], vy = uy[base + c];
      const double Tc = (numeq || ddf) ? (T ? T[base + c] : orc_phys_T0(g->phys)) : orc_phys_T0(g->phys);
      if (numeq) {
        /* start from the exponents of the continuous Maxwellian (numerical equilibrium) */
        const double PI = 3.14159265358979323846;
        lam[0] = (vx * vx + vy * vy) / (2.0 * Tc) + log(2.0 * PI * Tc) - 1.0;
        lam[1] = -vx / Tc; lam[2] = -vy / Tc; lam[3] = 1.0 / (2.0 * Tc); lam[4] = 0.0; lam[5] = 1.0 / (2.0 * Tc);
        lam[6] = 0.0; lam[7] = 0.0;
      }
      int it = orc_phys_equilibrium(g->phys, r, vx, vy, Tc, lam, feq, geq);
      double* s = L->S[0] + c * np;
      for (int i = 0; i < Q; ++i) s[i] = feq[i];
      if (ddf) for (int i = 0; i < Q; ++i) s[Q + i] = geq[i];
      if (numeq) for (int a = 0; a < ORC_NLAMBDA; ++a) s[loff + a] = lam[a];
      check_state(g, s, it);
    }
    memcpy(L->S[1], L->S[0], sizeof(double) * (size_t)(L->n * np));
    base += L->n;
  }
  for (int l = g->depth; l >= 1; --l) {
    orc_level* L = &g->lv[l];
    double f[ORC_QMAX], gg[ORC_QMAX], fo[ORC_QMAX], go[ORC_QMAX];
    for (int64_t q = 0; q < L->ng; ++q) {
      const int64_t c = L->g_coarse[q];
      double* s = L->S[L->cur] + c * np;
      for (int i = 0; i < Q; ++i) {
        const int unknown = (int)((L->g_mask[q] >> i) & 1ull);
        f[i] = unknown ? coalesce(g, l, q, i) : s[i];
        if (ddf) gg[i] = unknown ? coalesce(g, l, q, Q + i) : s[Q + i];
      }
      if (numeq) for (int a = 0; a < ORC_NLAMBDA; ++a) lam[a] = coalesce(g, l, q, loff + a);
      int it = orc_phys_collide(g->phys, L->tau, f, gg, lam, fo, go);
      for (int i = 0; i < Q; ++i) s[i] = fo[i];
      if (ddf) for (int i = 0; i < Q; ++i) s[Q + i] = go[i];
      if (numeq) for (int a = 0; a < ORC_NLAMBDA; ++a) s[loff + a] = lam[a];
      check_state(g, s, it);
      explode(g, l, q, s);
    }
  }
  return g->status;
}

int orc_get_macroscopic(const orc_grid* g, double* rho, double* ux, double* uy, double* T)
{
  int64_t base = 0;
  for (int l = 0; l <= g->depth; ++l) {
    const orc_level* L = &g->lv[l];
    const double* S = L->S[L->cur];
    for (int64_t c = 0; c < L->n; ++c) {
      double r, vx, vy, Tc;
      orc_phys_moments(g->phys, S + c * g->npop, S + c * g->npop + g->Q, &r, &vx, &vy, &Tc);
      if (rho) rho[base + c] = r;
      if (ux) ux[base + c] = vx;
      if (uy) uy[base + c] = vy;
      if (T) T[base + c] = Tc;
    }
    base += L->n;
  }
  return ORC_OK;
}

/* Refinement criterion of the paper's adaptive runs ("the kinetic sensor ... which basically evaluates the local
 * departure to equilibrium"): eps of Eq. 52, (1/V) sum_i |f_i - f_i^eq| / f_i^eq, of the CURRENT (post-collision) state
 * of every stored cell, f^eq = the model's equilibrium of the cell's own rho, u, T (numerical equilibria: solved from the
 * stored multipliers).  The collision of Eq. 30 scales f - f^eq by (1 - 1/tau_eff), so this is |1 - 1/tau_eff| times the eps
 * the last collision of the cell saw. */
int orc_get_sensor(orc_grid* g, double* eps)
{
  if (!g || !eps) return ORC_EINVAL;
  const int Q = g->Q;
  double feq[ORC_QMAX], geq[ORC_QMAX], lam[ORC_NLAMBDA];
  int64_t base = 0;
  for (int l = 0; l <= g->depth; ++l) {
    const orc_level* L = &g->lv[l];
    const double* S = L->S[L->cur];
    for (int64_t c = 0; c < L->n; ++c) {
      const double* f = S + c * g->npop;
      double r, vx, vy, Tc;
      orc_phys_moments(g->phys, f, f + Q, &r, &vx, &vy, &Tc);
      for (int k = 0; k < ORC_NLAMBDA; ++k) lam[k] = (g->cfg.collision == ORC_NUMEQ) ? f[(g->cfg.ddf ? 2 : 1) * Q + k] : 0.0;
      if (orc_phys_equilibrium(g->phys, r, vx, vy, Tc, lam, feq, geq) < 0) return ORC_ENEWTON;
      double e = 0.0;
      for (int i = 0; i < Q; ++i) {
        double den = fabs(feq[i]);
        if (den < 1e-300) den = 1e-300;
        e += fabs(f[i] - feq[i]) / den;
      }
      eps[base + c] = e / (double)Q;
    }
    base += L->n;
  }
  return ORC_OK;
}

static int pop_range(const orc_grid* g, int which, int* off, int* cnt)
{
  const int Q = g->Q, ddf = g->cfg.ddf, numeq = (g->cfg.collision == ORC_NUMEQ);
  if (which == 0) { *off = 0; *cnt = Q; return 0; }
  if (which == 1 && ddf) { *off = Q; *cnt = Q; return 0; }
  if (which == 2 && numeq) { *off = (ddf ? 2 : 1) * Q; *cnt = ORC_NLAMBDA; return 0; }
  return ORC_EINVAL;
}

/* position inside the coarse step (fine steps taken since its start), for tests that import a state taken mid-step */
int orc_set_fine_step(orc_grid* g, int64_t k)
{
  if (!g || k < 0) return ORC_EINVAL;
  g->k = k;
  return ORC_OK;
}

int orc_get_populations(const orc_grid* g, int l, int which, double* out)
{
  int off, cnt;
  if (l < 0 || l > g->depth || pop_range(g, which, &off, &cnt)) return ORC_EINVAL;
  const orc_level* L = &g->lv[l];
  const double* S = L->S[L->cur];
  for (int64_t c = 0; c < L->n; ++c)
    for (int p = 0; p < cnt; ++p) out[c * cnt + p] = S[c * g->npop + off + p];
  return ORC_OK;
}

int orc_set_populations(orc_grid* g, int l, int which, const double* in)
{
  int off, cnt;
  if (l < 0 || l > g->depth || pop_range(g, which, &off, &cnt)) return ORC_EINVAL;
  orc_level* L = &g->lv[l];
  double* S = L->S[L->cur];
  for (int64_t c = 0; c < L->n; ++c)
    for (int p = 0; p < cnt; ++p) S[c * g->npop + off + p] = in[c * cnt + p];
  return ORC_OK;
}
