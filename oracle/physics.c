/*
 * physics.c -- CPU ORACLE (test infrastructure): cell-local arithmetic.
 * Lattices (Table 4), Hermite polynomials (Eq. 35), polynomial
 * equilibria (Eq. 34, Table 5), recursive-regularised collision
 * (Eq. 33, 36-38 P:845-884), numerical equilibria (Eq. 39-49), second
 * distribution (Eq. 50-51), kinetic sensor (Eq. 52-53).
 * Plain fp64, canonical direction order, sums left to right.  No code is shared with
 * the CUDA path.
 */
#include "oracle.h"
#include <math.h>
#include <string.h>
#include <stdlib.h>

/* ------------------------------------------------------------------ lattices */

typedef struct {
  int Q, W;
  double cs2;
  int cx[ORC_QMAX], cy[ORC_QMAX], opp[ORC_QMAX];
  double w[ORC_QMAX];
  int use3_full;  /* xxx, yyy in the basis (Table 5) */
  int use3_mixed; /* xxy, xyy */
  int use4_xxyy;  /* xxyy */
  int use4_full;  /* xxxx, xxxy, xyyy, yyyy */
} lat_t;

/* groups of Table 4 in row order: (0,0) (1,0) (1,1) (2,0) (2,1) (2,2) (3,0) (3,1) */
static const int GRP_A[8] = {0, 1, 1, 2, 2, 2, 3, 3};
static const int GRP_B[8] = {0, 0, 1, 0, 1, 2, 0, 1};

static int push_group(lat_t* L, int n, int a, int b, double w)
{
  /* canonical order inside a group: counter-clockwise from the +x axis */
  if (a == 0 && b == 0) { L->cx[n] = 0; L->cy[n] = 0; L->w[n] = w; return n + 1; }
  if (b == 0) {
    const int X[4] = {a, 0, -a, 0}, Y[4] = {0, a, 0, -a};
    for (int k = 0; k < 4; ++k) { L->cx[n] = X[k]; L->cy[n] = Y[k]; L->w[n] = w; ++n; }
    return n;
  }
  if (a == b) {
    const int X[4] = {a, -a, -a, a}, Y[4] = {a, a, -a, -a};
    for (int k = 0; k < 4; ++k) { L->cx[n] = X[k]; L->cy[n] = Y[k]; L->w[n] = w; ++n; }
    return n;
  }
  {
    const int X[8] = {a, b, -b, -a, -a, -b, b, a}, Y[8] = {b, a, a, b, -b, -a, -a, -b};
    for (int k = 0; k < 8; ++k) { L->cx[n] = X[k]; L->cy[n] = Y[k]; L->w[n] = w; ++n; }
    return n;
  }
}

static int lat_build(int Q, lat_t* L)
{
  double wg[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  int present[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  memset(L, 0, sizeof(*L));
  switch (Q) {
  case 9:  /* Table 4 column D2Q9 */
    wg[0] = 4.0 / 9.0; wg[1] = 1.0 / 9.0; wg[2] = 1.0 / 36.0;
    present[0] = present[1] = present[2] = 1;
    L->cs2 = 1.0 / 3.0; L->W = 1;
    L->use3_mixed = 1; L->use4_xxyy = 1;           /* Table 5: partial 4th order */
    break;
  case 13: /* D2Q13 */
    wg[0] = 36.0 / 96.0; wg[1] = 8.0 / 96.0; wg[2] = 6.0 / 96.0; wg[3] = 1.0 / 96.0;
    present[0] = present[1] = present[2] = present[3] = 1;
    L->cs2 = 1.0 / 2.0; L->W = 2;
    L->use3_full = 1; L->use3_mixed = 1;           /* full 3rd order */
    break;
  case 21: /* D2Q21 */
    wg[0] = 91.0 / 324.0; wg[1] = 1.0 / 12.0; wg[2] = 2.0 / 27.0; wg[3] = 7.0 / 360.0;
    wg[5] = 1.0 / 432.0; wg[6] = 1.0 / 1620.0;
    present[0] = present[1] = present[2] = present[3] = present[5] = present[6] = 1;
    L->cs2 = 2.0 / 3.0; L->W = 3;
    L->use3_full = 1; L->use3_mixed = 1;
    break;
  case 37: /* D2Q37, 15-digit decimals verbatim (S23) */
    wg[0] = 0.233150669132352; wg[1] = 0.107306091542219; wg[2] = 0.057667859888794;
    wg[3] = 0.014208216158450; wg[4] = 0.005353049000513; wg[5] = 0.001011937592673;
    wg[6] = 0.000245301027757; wg[7] = 0.000283414252994;
    for (int k = 0; k < 8; ++k) present[k] = 1;
    L->cs2 = 0.697953322019683; L->W = 3;
    L->use3_full = 1; L->use3_mixed = 1; L->use4_xxyy = 1; L->use4_full = 1;  /* full 4th order */
    break;
  default:
    return ORC_EINVAL;
  }
  int n = 0;
  for (int k = 0; k < 8; ++k)
    if (present[k]) n = push_group(L, n, GRP_A[k], GRP_B[k], wg[k]);
  L->Q = n;
  if (n != Q) return ORC_EINVAL;
  for (int i = 0; i < Q; ++i) {
    L->opp[i] = -1;
    for (int j = 0; j < Q; ++j)
      if (L->cx[j] == -L->cx[i] && L->cy[j] == -L->cy[i]) L->opp[i] = j;
  }
  return ORC_OK;
}

int orc_lattice(int Q, int* cx, int* cy, double* w, int* opp, double* cs2, int* reach)
{
  lat_t L;
  int rc = lat_build(Q, &L);
  if (rc) return rc;
  for (int i = 0; i < Q; ++i) {
    if (cx) cx[i] = L.cx[i];
    if (cy) cy[i] = L.cy[i];
    if (w) w[i] = L.w[i];
    if (opp) opp[i] = L.opp[i];
  }
  if (cs2) *cs2 = L.cs2;
  if (reach) *reach = L.W;
  return ORC_OK;
}

/* --------------------------------------------------- Hermite moment vectors */
/* 15 components: 0 | x y | xx xy yy | xxx xxy xyy yyy | xxxx xxxy xxyy xyyy yyyy */
enum { A0 = 0, AX, AY, AXX, AXY, AYY, AXXX, AXXY, AXYY, AYYY, AXXXX, AXXXY, AXXYY, AXYYY, AYYYY, NA };

/* Eq. 36 (athermal) and its thermal generalisation (reading "thermal moments"):
 * Hermite moments of a Maxwellian of temperature T about T0 = c_s^2, th = T - c_s^2. */
static void aeq_moments(double rho, double ux, double uy, double th, double* a)
{
  a[A0] = rho;
  a[AX] = rho * ux;
  a[AY] = rho * uy;
  a[AXX] = rho * (ux * ux + th);
  a[AXY] = rho * (ux * uy);
  a[AYY] = rho * (uy * uy + th);
  a[AXXX] = rho * (ux * ux * ux + 3.0 * th * ux);
  a[AXXY] = rho * (ux * ux * uy + th * uy);
  a[AXYY] = rho * (ux * uy * uy + th * ux);
  a[AYYY] = rho * (uy * uy * uy + 3.0 * th * uy);
  a[AXXXX] = rho * (ux * ux * ux * ux + 6.0 * th * ux * ux + 3.0 * th * th);
  a[AXXXY] = rho * (ux * ux * ux * uy + 3.0 * th * ux * uy);
  a[AXXYY] = rho * (ux * ux * uy * uy + th * (ux * ux + uy * uy) + th * th);
  a[AXYYY] = rho * (ux * uy * uy * uy + 3.0 * th * ux * uy);
  a[AYYYY] = rho * (uy * uy * uy * uy + 6.0 * th * uy * uy + 3.0 * th * th);
}

/* Eq. 33 / 34: f_i = w_i sum_n 1/(n! cs^2n) H_i^(n) : a^(n), restricted to the basis of
 * Table 5.  The full contraction counts xy twice, xxy/xyy three times, xxxy/xyyy four
 * times and xxyy six times. */
static void poly_from_moments(const lat_t* L, const double* a, double* f)
{
  const double c2 = L->cs2, c4 = c2 * c2, c6 = c4 * c2, c8 = c4 * c4;
  for (int i = 0; i < L->Q; ++i) {
    const double x = L->cx[i], y = L->cy[i];
    /* Eq. 35 */
    const double Hxx = x * x - c2, Hyy = y * y - c2, Hxy = x * y;
    const double Hxxx = (x * x - 3.0 * c2) * x, Hyyy = (y * y - 3.0 * c2) * y;
    const double Hxxy = (x * x - c2) * y, Hxyy = (y * y - c2) * x;
    const double Hxxxx = x * x * x * x - 6.0 * c2 * x * x + 3.0 * c4;
    const double Hyyyy = y * y * y * y - 6.0 * c2 * y * y + 3.0 * c4;
    const double Hxxxy = (x * x - 3.0 * c2) * x * y, Hxyyy = (y * y - 3.0 * c2) * y * x;
    const double Hxxyy = (x * x - c2) * (y * y - c2);
    double s = a[A0];
    s += (x * a[AX] + y * a[AY]) / c2;
    s += (Hxx * a[AXX] + 2.0 * Hxy * a[AXY] + Hyy * a[AYY]) / (2.0 * c4);
    double s3 = 0.0;
    if (L->use3_full) s3 += Hxxx * a[AXXX] + Hyyy * a[AYYY];
    if (L->use3_mixed) s3 += 3.0 * Hxxy * a[AXXY] + 3.0 * Hxyy * a[AXYY];
    s += s3 / (6.0 * c6);
    double s4 = 0.0;
    if (L->use4_full) s4 += Hxxxx * a[AXXXX] + Hyyyy * a[AYYYY] + 4.0 * Hxxxy * a[AXXXY] + 4.0 * Hxyyy * a[AXYYY];
    if (L->use4_xxyy) s4 += 6.0 * Hxxyy * a[AXXYY];
    s += s4 / (24.0 * c8);
    f[i] = L->w[i] * s;
  }
}

static void feq_poly(const lat_t* L, double rho, double ux, double uy, double T, int thermal, double* feq)
{
  double a[NA];
  aeq_moments(rho, ux, uy, thermal ? (T - L->cs2) : 0.0, a);
  poly_from_moments(L, a, feq);
}

int orc_feq_poly(int Q, double rho, double ux, double uy, double T, int thermal, double* feq)
{
  lat_t L;
  int rc = lat_build(Q, &L);
  if (rc) return rc;
  feq_poly(&L, rho, ux, uy, T, thermal, feq);
  return ORC_OK;
}

/* ------------------------------------------------------ numerical equilibrium */
/* monomials paired with the 8 multipliers: 1, x, y, xx, xy, yy, x(xx+yy), y(xx+yy)  (Eq. 42-49) */
static void monomials(const lat_t* L, double M[ORC_QMAX][ORC_NLAMBDA])
{
  for (int i = 0; i < L->Q; ++i) {
    const double x = L->cx[i], y = L->cy[i], r2 = x * x + y * y;
    M[i][0] = 1.0; M[i][1] = x; M[i][2] = y; M[i][3] = x * x; M[i][4] = x * y; M[i][5] = y * y;
    M[i][6] = x * r2; M[i][7] = y * r2;
  }
}

/* f_i(lambda) = rho exp[-(1 + sum_a lambda_a M_ia)] (Eq. 39 with a = rho);
 * G_a = sum_i f_i M_ia - m_a (Eq. 42-49) */
static void numeq_eval(const lat_t* L, double M[ORC_QMAX][ORC_NLAMBDA], double rho, const double* m,
                       const double* lam, double* f, double* G)
{
  for (int a = 0; a < ORC_NLAMBDA; ++a) G[a] = 0.0;
  for (int i = 0; i < L->Q; ++i) {
    double e = 1.0;
    for (int a = 0; a < ORC_NLAMBDA; ++a) e += lam[a] * M[i][a];
    f[i] = rho * exp(-e);
    for (int a = 0; a < ORC_NLAMBDA; ++a) G[a] += f[i] * M[i][a];
  }
  for (int a = 0; a < ORC_NLAMBDA; ++a) G[a] -= m[a];
}

/* solve (-J) d = G with -J = sum_i f_i M_i M_i^T symmetric positive definite, by Cholesky.
 * returns 0 on success */
static int newton_direction(const lat_t* L, double M[ORC_QMAX][ORC_NLAMBDA], const double* f, const double* G, double* d)
{
  double A[ORC_NLAMBDA][ORC_NLAMBDA];
  for (int a = 0; a < ORC_NLAMBDA; ++a)
    for (int b = 0; b < ORC_NLAMBDA; ++b) {
      double s = 0.0;
      for (int i = 0; i < L->Q; ++i) s += f[i] * M[i][a] * M[i][b];
      A[a][b] = s;
    }
  /* A = C C^T */
  double C[ORC_NLAMBDA][ORC_NLAMBDA];
  memset(C, 0, sizeof(C));
  for (int j = 0; j < ORC_NLAMBDA; ++j) {
    double s = A[j][j];
    for (int k = 0; k < j; ++k) s -= C[j][k] * C[j][k];
    if (!(s > 0.0)) return 1;
    C[j][j] = sqrt(s);
    for (int i = j + 1; i < ORC_NLAMBDA; ++i) {
      double t = A[i][j];
      for (int k = 0; k < j; ++k) t -= C[i][k] * C[j][k];
      C[i][j] = t / C[j][j];
    }
  }
  double y[ORC_NLAMBDA];
  for (int i = 0; i < ORC_NLAMBDA; ++i) {
    double t = G[i];
    for (int k = 0; k < i; ++k) t -= C[i][k] * y[k];
    y[i] = t / C[i][i];
  }
  for (int i = ORC_NLAMBDA - 1; i >= 0; --i) {
    double t = y[i];
    for (int k = i + 1; k < ORC_NLAMBDA; ++k) t -= C[k][i] * d[k];
    d[i] = t / C[i][i];
  }
  /* J d = -G  with J = -A  =>  A d = G, so lambda_new = lambda + d */
  return 0;
}

static double norm2(const double* G)
{
  double s = 0.0;
  for (int a = 0; a < ORC_NLAMBDA; ++a) s += G[a] * G[a];
  return sqrt(s);
}

/* Newton-Raphson with a halving line search (stopping rule: DESIGN.md S14):
 * iterate until sum|G_a| <= tol*rho or max_iter, then one unconditional full Newton step.
 * returns the number of Newton steps taken (polish included), negative if not converged
 * or if the Jacobian is not positive definite. */
static int feq_numerical(const lat_t* L, double rho, double ux, double uy, double T, double tol, int max_iter,
                         double* lam, double* feq)
{
  double M[ORC_QMAX][ORC_NLAMBDA];
  monomials(L, M);
  const double u2 = ux * ux + uy * uy;
  /* right-hand sides of Eq. 42-49 with 2E = u^2 + 2T  =>  2(E+T) = u^2 + 4T */
  const double m[ORC_NLAMBDA] = {rho, rho * ux, rho * uy, rho * (ux * ux + T), rho * ux * uy, rho * (uy * uy + T),
                                 rho * ux * (u2 + 4.0 * T), rho * uy * (u2 + 4.0 * T)};
  double f[ORC_QMAX], G[ORC_NLAMBDA], d[ORC_NLAMBDA], lt[ORC_NLAMBDA], ft[ORC_QMAX], Gt[ORC_NLAMBDA];
  int it = 0, converged = 0, bad = 0;
  numeq_eval(L, M, rho, m, lam, f, G);
  for (;;) {
    double r1 = 0.0;
    for (int a = 0; a < ORC_NLAMBDA; ++a) r1 += fabs(G[a]);
    if (r1 <= tol * rho) { converged = 1; break; }
    if (it >= max_iter) break;
    if (newton_direction(L, M, f, G, d)) { bad = 1; break; }
    const double n0 = norm2(G);
    double t = 1.0;
    for (;;) {
      for (int a = 0; a < ORC_NLAMBDA; ++a) lt[a] = lam[a] + t * d[a];
      numeq_eval(L, M, rho, m, lt, ft, Gt);
      const double n1 = norm2(Gt);
      if (n1 < n0 || t <= 1.0 / 1024.0) break;   /* NaN n1 fails the first test and keeps halving */
      t *= 0.5;
    }
    for (int a = 0; a < ORC_NLAMBDA; ++a) lam[a] = lt[a];
    memcpy(f, ft, sizeof(double) * L->Q);
    memcpy(G, Gt, sizeof(G));
    ++it;
  }
  if (!bad) { /* polish: one further full Newton step, unconditionally */
    if (newton_direction(L, M, f, G, d) == 0) {
      for (int a = 0; a < ORC_NLAMBDA; ++a) lam[a] += d[a];
      numeq_eval(L, M, rho, m, lam, f, G);
      ++it;
    } else bad = 1;
  }
  memcpy(feq, f, sizeof(double) * L->Q);
  return (converged && !bad) ? it : -it - 1;
}

int orc_feq_numerical(int Q, double rho, double ux, double uy, double T, double tol, int max_iter,
                      double* lambda, double* feq)
{
  lat_t L;
  int rc = lat_build(Q, &L);
  if (rc) return -1000;
  return feq_numerical(&L, rho, ux, uy, T, tol, max_iter, lambda, feq);
}

/* ------------------------------------------------------------- one collision */

/* Eq. 53 with the reading S10: alpha = 1 below 0.01; third case alpha = 1/tau */
static double sensor_alpha(double eps, double A, double tau)
{
  if (eps < 0.01) return 1.0;
  if (eps < 0.10) return 1.05;
  if (eps < 1.00) return A;
  return 1.0 / tau;
}

typedef struct phys_t {
  lat_t L;
  orc_config cfg;
} phys_t;

int orc_phys_init(phys_t* P, const orc_config* cfg)
{
  int rc = lat_build(cfg->lattice, &P->L);
  if (rc) return rc;
  P->cfg = *cfg;
  if (cfg->collision != ORC_NUMEQ) P->cfg.T0 = P->L.cs2;
  if (cfg->collision == ORC_RR && cfg->ddf) return ORC_EINVAL;  /* RR is defined for the athermal models only */
  if (cfg->collision < 0 || cfg->collision > 2) return ORC_EINVAL;
  return ORC_OK;
}

/* macroscopic moments of a population set: rho, u (a2), T (Eq. 51, or T0 for athermal models) */
void orc_phys_moments(const phys_t* P, const double* f, const double* g, double* rho, double* ux, double* uy, double* T)
{
  const lat_t* L = &P->L;
  double r = 0.0, jx = 0.0, jy = 0.0;
  for (int i = 0; i < L->Q; ++i) { r += f[i]; jx += L->cx[i] * f[i]; jy += L->cy[i] * f[i]; }
  const double vx = jx / r, vy = jy / r;
  *rho = r; *ux = vx; *uy = vy;
  const int thermal = (P->cfg.collision == ORC_NUMEQ) || P->cfg.ddf;
  if (!thermal) { *T = P->cfg.T0; return; }
  /* Eq. 51: T = [sum_i (xi^2 f_i + g_i) - rho u^2] / (2 rho C_v); C_v = 1/(gamma-1), or D/2 = 1 without g */
  double e2 = 0.0;
  for (int i = 0; i < L->Q; ++i) {
    const double xi2 = (double)(L->cx[i] * L->cx[i] + L->cy[i] * L->cy[i]);
    e2 += xi2 * f[i] + (P->cfg.ddf ? g[i] : 0.0);
  }
  const double Cv = P->cfg.ddf ? 1.0 / (P->cfg.gamma - 1.0) : 1.0;
  *T = (e2 - r * (vx * vx + vy * vy)) / (2.0 * r * Cv);
}

/* equilibrium of the configured model for given macroscopic state; lambda in/out for NUMEQ.
 * returns Newton iterations (0 for polynomial), negative on failure */
int orc_phys_equilibrium(const phys_t* P, double rho, double ux, double uy, double T, double* lam, double* feq, double* geq)
{
  const lat_t* L = &P->L;
  int it = 0;
  if (P->cfg.collision == ORC_NUMEQ)
    it = feq_numerical(L, rho, ux, uy, T, P->cfg.newton_tol, P->cfg.newton_max_iter, lam, feq);
  else
    feq_poly(L, rho, ux, uy, T, P->cfg.ddf, feq);
  if (P->cfg.ddf) {
    const double Cv = 1.0 / (P->cfg.gamma - 1.0);
    const double fac = (2.0 * Cv - 2.0) * T;      /* Eq. 50, D = 2 */
    for (int i = 0; i < L->Q; ++i) geq[i] = fac * feq[i];
  }
  return it;
}

/* steps 2-5 of the cell update: moments, equilibrium, sensor, relaxation */
int orc_phys_collide(const phys_t* P, double tau, const double* f, const double* g, double* lam, double* fout, double* gout)
{
  const lat_t* L = &P->L;
  const int Q = L->Q;
  double rho, ux, uy, T;
  double feq[ORC_QMAX], geq[ORC_QMAX];
  orc_phys_moments(P, f, g, &rho, &ux, &uy, &T);
  int it = orc_phys_equilibrium(P, rho, ux, uy, T, lam, feq, geq);
  double tau_eff = tau;
  if (P->cfg.sensor) {
    double eps = 0.0;
    for (int i = 0; i < Q; ++i) {
      double den = fabs(feq[i]);
      if (den < 1e-300) den = 1e-300;
      eps += fabs(f[i] - feq[i]) / den;           /* Eq. 52 */
    }
    eps /= (double)Q;
    tau_eff = tau * sensor_alpha(eps, P->cfg.sensor_A, tau);
  }
  const double keep = 1.0 - 1.0 / tau_eff;
  if (P->cfg.collision == ORC_RR) {
    /* Pi = sum_i H_i^(2) (f_i - f_i^eq) */
    const double c2 = L->cs2;
    double pxx = 0.0, pxy = 0.0, pyy = 0.0;
    for (int i = 0; i < Q; ++i) {
      const double x = L->cx[i], y = L->cy[i], dn = f[i] - feq[i];
      pxx += (x * x - c2) * dn; pxy += (x * y) * dn; pyy += (y * y - c2) * dn;
    }
    if (P->cfg.trace_eq) { /* trace relaxes with tau = 1: only the deviatoric part survives (S7) */
      const double dev = 0.5 * (pxx - pyy);
      pxx = dev; pyy = -dev;
    }
    double an[NA], ae[NA], as[NA];
    memset(an, 0, sizeof(an));
    an[AXX] = pxx; an[AXY] = pxy; an[AYY] = pyy;
    /* Eq. 37-38 (with the typo of P:876 repaired, S2) */
    an[AXXX] = 3.0 * ux * pxx;
    an[AXXY] = 2.0 * ux * pxy + uy * pxx;
    an[AXYY] = 2.0 * uy * pxy + ux * pyy;
    an[AYYY] = 3.0 * uy * pyy;
    an[AXXXX] = 4.0 * ux * an[AXXX] - 6.0 * ux * ux * pxx;
    an[AXXXY] = (3.0 * ux * an[AXXY] + uy * an[AXXX]) - 3.0 * ux * ux * pxy - 3.0 * ux * uy * pxx;
    an[AXXYY] = 2.0 * (ux * an[AXYY] + uy * an[AXXY]) - ux * ux * pyy - uy * uy * pxx - 4.0 * ux * uy * pxy;
    an[AXYYY] = (3.0 * uy * an[AXYY] + ux * an[AYYY]) - 3.0 * uy * uy * pxy - 3.0 * ux * uy * pyy;
    an[AYYYY] = 4.0 * uy * an[AYYY] - 6.0 * uy * uy * pyy;
    aeq_moments(rho, ux, uy, 0.0, ae);
    for (int k = 0; k < NA; ++k) as[k] = ae[k] + keep * an[k];   /* a* = a_eq + (1-1/tau) a_neq */
    poly_from_moments(L, as, fout);                               /* Eq. 33 */
  } else {
    for (int i = 0; i < Q; ++i) fout[i] = feq[i] + keep * (f[i] - feq[i]);     /* Eq. 30 */
  }
  if (P->cfg.ddf)
    for (int i = 0; i < Q; ++i) gout[i] = geq[i] + keep * (g[i] - geq[i]);
  return it;
}

int orc_collide_cell(const orc_config* cfg, double tau, const double* f, const double* g,
                     double* lambda, double* fout, double* gout)
{
  phys_t P;
  int rc = orc_phys_init(&P, cfg);
  if (rc) return -1000;
  return orc_phys_collide(&P, tau, f, g, lambda, fout, gout);
}

/* accessors used by sim.c (kept here so that lat_t stays private to this file) */
int orc_phys_Q(const phys_t* P) { return P->L.Q; }
int orc_phys_W(const phys_t* P) { return P->L.W; }
int orc_phys_cx(const phys_t* P, int i) { return P->L.cx[i]; }
int orc_phys_cy(const phys_t* P, int i) { return P->L.cy[i]; }
int orc_phys_opp(const phys_t* P, int i) { return P->L.opp[i]; }
double orc_phys_w(const phys_t* P, int i) { return P->L.w[i]; }
double orc_phys_cs2(const phys_t* P) { return P->L.cs2; }
double orc_phys_T0(const phys_t* P) { return P->cfg.T0; }
phys_t* orc_phys_new(const orc_config* cfg, int* rc)
{
  phys_t* P = (phys_t*)calloc(1, sizeof(phys_t));
  if (!P) { *rc = ORC_ENOMEM; return 0; }
  *rc = orc_phys_init(P, cfg);
  if (*rc) { free(P); return 0; }
  return P;
}
