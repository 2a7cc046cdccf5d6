// collide.cuh -- cell-local arithmetic of the CUDA path (rows a2-a5 of SURVEY.md Sec. 8(a)):
// moments, polynomial equilibria (Eq. 34-36), recursive-regularised collision
// (Eq. 33, 37-38 P:845-884), numerical equilibria (Eq. 39-49), second distribution
// (Eq. 50-51), kinetic sensor (Eq. 52-53), BGK relaxation (Eq. 30).
// Everything stays in registers; lattice constants are compile-time immediates (lattice.cuh).
#pragma once
#include <cuda_runtime.h>

#include "../../include/lbm.h"
#include "lattice.cuh"

namespace lbm {

// Model constants, passed to every kernel by value.
struct ModelParams {
  double gamma, sensor_A, T0, newton_tol;
  int newton_max_iter, trace_eq;
  int bc_kind[4];
  double bc_rho[4], bc_ux[4], bc_uy[4], bc_T[4];
  double sponge_rho_inf;
};

enum { FLAG_UNSTABLE = 1, FLAG_NEWTON = 2 };

// 1/x to within ~1 ulp for normal x: hardware seed (MUFU.RCP64H, ~20 bits) + two Newton steps (4 DFMA) instead
// of the IEEE division routine (~25 instructions and a call); used where Q quotients per cell are summed (Eq. 52).
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}
__device__ __forceinline__ float fast_rcp(float x) { return 1.0f / x; }
__device__ __forceinline__ void opaque(double& x) { asm volatile("" : "+d"(x)); }
__device__ __forceinline__ void opaque(float& x) { asm volatile("" : "+f"(x)); }

template <typename T> struct Num;
template <> struct Num<double> {
  static __device__ __forceinline__ double tiny() { return 1e-300; }
  static __device__ __forceinline__ double exp_(double x) { return exp(x); }
  static __device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
  static __device__ __forceinline__ double abs_(double x) { return fabs(x); }
};
template <> struct Num<float> {
  static __device__ __forceinline__ float tiny() { return 1e-37f; }
  static __device__ __forceinline__ float exp_(float x) { return expf(x); }
  static __device__ __forceinline__ float sqrt_(float x) { return sqrtf(x); }
  static __device__ __forceinline__ float abs_(float x) { return fabsf(x); }
};

// Hermite moments of the equilibrium: Eq. 36 (athermal, th = 0) and their thermal generalisation
// about T0 = c_s^2, th = T - c_s^2 (the paper prints only the athermal ones).
template <typename T>
__device__ __forceinline__ void aeq_moments(T rho, T ux, T uy, T th, T (&a)[NA]) {
  const T ux2 = ux * ux, uy2 = uy * uy;
  a[A0] = rho;
  a[AX] = rho * ux;
  a[AY] = rho * uy;
  a[AXX] = rho * (ux2 + th);
  a[AXY] = rho * (ux * uy);
  a[AYY] = rho * (uy2 + th);
  a[AXXX] = rho * (ux2 * ux + T(3) * th * ux);
  a[AXXY] = rho * (ux2 * uy + th * uy);
  a[AXYY] = rho * (ux * uy2 + th * ux);
  a[AYYY] = rho * (uy2 * uy + T(3) * th * uy);
  a[AXXXX] = rho * (ux2 * ux2 + T(6) * th * ux2 + T(3) * th * th);
  a[AXXXY] = rho * (ux2 * ux * uy + T(3) * th * ux * uy);
  a[AXXYY] = rho * (ux2 * uy2 + th * (ux2 + uy2) + th * th);
  a[AXYYY] = rho * (ux * uy2 * uy + T(3) * th * ux * uy);
  a[AYYYY] = rho * (uy2 * uy2 + T(6) * th * uy2 + T(3) * th * th);
}

// f_i of Eq. 33/34 from the Hermite moments a, restricted to the basis of Table 5.
template <int Q, typename T, int I>
__device__ __forceinline__ T poly_i(const T (&a)[NA]) {
  constexpr double c0 = hermite_coef(Lat<Q>::t, I, A0);
  T s = T(c0) * a[A0];
  static_for<1, NA>([&](auto kc) {
    constexpr int K = decltype(kc)::value;
    constexpr double c = hermite_coef(Lat<Q>::t, I, K);
    if constexpr (c != 0.0) s += T(c) * a[K];
  });
  return s;
}

// Order of the Hermite moment in slot k (parity decides the sign under xi -> -xi).
__host__ __device__ constexpr int slot_order(int k) { return k == A0 ? 0 : k <= AY ? 1 : k <= AYY ? 2 : k <= AYYY ? 3 : 4; }

// f_I and f_opp(I) of Eq. 33/34 together: the even-order part is shared, the odd-order part changes sign
// (H^(n)(-xi) = (-1)^n H^(n)(xi), w_opp = w), which halves the multiply-adds of the reconstruction.
template <int Q, typename T, int I>
__device__ __forceinline__ void poly_pair(const T (&a)[NA], T& fi, T& fo) {
  constexpr double c0 = hermite_coef(Lat<Q>::t, I, A0);
  T e = T(c0) * a[A0], o = T(0);
  static_for<1, NA>([&](auto kc) {
    constexpr int K = decltype(kc)::value;
    constexpr double c = hermite_coef(Lat<Q>::t, I, K);
    if constexpr (c != 0.0) {
      if constexpr (slot_order(K) % 2 == 1) o += T(c) * a[K];
      else e += T(c) * a[K];
    }
  });
  fi = e + o;
  fo = e - o;
}

// fn(I, fe_I) for every direction, evaluated pairwise
template <int Q, typename T, class F>
__device__ __forceinline__ void poly_all(const T (&a)[NA], F&& fn) {
  fn(std::integral_constant<int, 0>{}, poly_i<Q, T, 0>(a));
  static_for<1, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int O = Lat<Q>::t.opp[I];
    if constexpr (O > I) {
      T fi, fo;
      poly_pair<Q, T, I>(a, fi, fo);
      fn(std::integral_constant<int, I>{}, fi);
      fn(std::integral_constant<int, O>{}, fo);
    }
  });
}

// rho, u (a2) and T by Eq. 51 (thermal models) or T0 = c_s^2 (athermal)
template <int Q, typename T, bool THERMAL, bool DDF>
__device__ __forceinline__ void moments(const ModelParams& p, const T (&f)[Q], const T (&g)[Q], T& rho, T& ux, T& uy, T& Tm) {
  T r = T(0), jx = T(0), jy = T(0);
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I];
    r += f[I];
    if constexpr (cx != 0) jx += T(cx) * f[I];
    if constexpr (cy != 0) jy += T(cy) * f[I];
  });
  rho = r; ux = jx / r; uy = jy / r;
  if constexpr (!THERMAL) {
    Tm = T(cs2_v<Q>);
  } else {
    T e2 = T(0);
    static_for<0, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      constexpr int xi2 = Lat<Q>::t.cx[I] * Lat<Q>::t.cx[I] + Lat<Q>::t.cy[I] * Lat<Q>::t.cy[I];
      if constexpr (DDF) e2 += T(xi2) * f[I] + g[I];
      else if constexpr (xi2 != 0) e2 += T(xi2) * f[I];
    });
    const T Cv = DDF ? T(1.0 / (p.gamma - 1.0)) : T(1);
    Tm = (e2 - r * (ux * ux + uy * uy)) / (T(2) * r * Cv);
  }
}

// ------------------------------------------------------------------ numerical equilibrium
__host__ __device__ constexpr int ipow_c(int b, int e) { int r = 1; for (int k = 0; k < e; ++k) r *= b; return r; }

// x^N for a compile-time N >= 0 by binary exponentiation (identical sub-powers are shared by the compiler)
template <int N, typename T>
__device__ __forceinline__ T ipow(T x) {
  if constexpr (N == 0) return T(1);
  else if constexpr (N == 1) return x;
  else if constexpr (N % 2 == 0) { const T h = ipow<N / 2, T>(x); return h * h; }
  else return ipow<N - 1, T>(x) * x;
}

// Reflection combinations.  Every lattice of Table 4 is symmetric under x -> -x and under y -> -y, and every sum the solver
// needs is a moment sum_i f_i x^PX y^PY (x^2 + y^2)^PR, which sees only the part of f that is even / odd in x and in y
// according to the parities of PX and PY.  So the Q values are first combined per reflection orbit -- (a, b), a, b > 0:
// EE, OE, EO, OO by a two-stage butterfly (8 additions); (a, 0) and (0, b): E, O (2 additions) -- and each moment is then ONE
// multiply-add per orbit instead of one per direction: D2Q21's 8 residual sums + 16 Jacobian sums take 28 + 41 + 56
// instructions instead of 113 + 176.  The combination lives in the slot of the orbit member whose signs spell its parities
// (x < 0: odd in x, y < 0: odd in y).  Only the order of the additions differs from the plain sums.
// fp64 only: in fp32 the D2Q37 solve sits on its rounding floor (tolerance 1e-5 of P:934 against ~1e-6 rho of summation
// noise amplified by the Jacobian): re-forming these sums, in this or in any other order, moved the worst cell of the
// 48^2 parity case from 1.5e-6 to 3.5e-5 of the oracle, so the fp32 kernels keep the plain sums, interleaved with the
// evaluation of f exactly as before (plain_moment below).
template <typename T> constexpr bool USE_REFLECT_COMBOS = sizeof(T) == 8;

__host__ __device__ constexpr int dir_index(const LatTab& L, int x, int y) {
  for (int i = 0; i < L.Q; ++i)
    if (L.cx[i] == x && L.cy[i] == y) return i;
  return -1;
}

template <int Q, typename T>
__device__ __forceinline__ void reflect_combos(const T (&f)[Q], T (&s)[Q]) {
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int x = Lat<Q>::t.cx[I], y = Lat<Q>::t.cy[I];
    if constexpr (x == 0 && y == 0) {
      s[I] = f[I];
    } else if constexpr ((x > 0 && y == 0) || (x == 0 && y > 0)) {
      constexpr int J = dir_index(Lat<Q>::t, -x, -y);
      static_assert(J >= 0, "lattice is not reflection-symmetric");
      s[I] = f[I] + f[J];
      s[J] = f[I] - f[J];
    } else if constexpr (x > 0 && y > 0) {
      constexpr int Jx = dir_index(Lat<Q>::t, -x, y), Jy = dir_index(Lat<Q>::t, x, -y), Jxy = dir_index(Lat<Q>::t, -x, -y);
      static_assert(Jx >= 0 && Jy >= 0 && Jxy >= 0, "lattice is not reflection-symmetric");
      const T p1 = f[I] + f[Jx], m1 = f[I] - f[Jx];      // y = +b row: even / odd in x
      const T p2 = f[Jy] + f[Jxy], m2 = f[Jy] - f[Jxy];  // y = -b row
      s[I] = p1 + p2;      // EE
      s[Jx] = m1 + m2;     // odd in x, even in y
      s[Jy] = p1 - p2;     // even in x, odd in y
      s[Jxy] = m1 - m2;    // OO
    }
  });
}

// sum_i f_i x_i^PX y_i^PY (x_i^2 + y_i^2)^PR from the reflection combinations s of f
template <int Q, typename T, int PX, int PY, int PR>
__device__ __forceinline__ T sym_moment(const T (&s)[Q]) {
  T acc = T(0);
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int x = Lat<Q>::t.cx[I], y = Lat<Q>::t.cy[I];
    constexpr int ax = x < 0 ? -x : x, ay = y < 0 ? -y : y;
    constexpr bool match = ((PX & 1) == (x < 0 ? 1 : 0)) && ((PY & 1) == (y < 0 ? 1 : 0));
    constexpr int wgt = ipow_c(ax, PX) * ipow_c(ay, PY) * ipow_c(x * x + y * y, PR);
    if constexpr (match && wgt != 0) acc += s[I] * T(wgt);
  });
  return acc;
}

// sum_i f_i x_i^PX y_i^PY (x_i^2 + y_i^2)^PR over the directions where the weight is not zero (fp32 kernels)
template <int Q, typename T, int PX, int PY, int PR>
__device__ __forceinline__ T plain_moment(const T (&f)[Q]) {
  T s = T(0);
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int x = Lat<Q>::t.cx[I], y = Lat<Q>::t.cy[I];
    constexpr int wgt = ipow_c(x, PX) * ipow_c(y, PY) * ipow_c(x * x + y * y, PR);
    if constexpr (wgt != 0) s += f[I] * T(wgt);
  });
  return s;
}

// the moment from whichever form the precision uses: s = reflection combinations (fp64) or f itself (fp32)
template <int Q, typename T, int PX, int PY, int PR>
__device__ __forceinline__ T solver_moment(const T (&s)[Q]) {
  if constexpr (USE_REFLECT_COMBOS<T>) return sym_moment<Q, T, PX, PY, PR>(s);
  else return plain_moment<Q, T, PX, PY, PR>(s);
}

// f_i(lambda) = rho exp[-(1 + sum_a lambda_a M_ia)] (Eq. 39 with a = rho); G_a = sum_i f_i M_ia - m_a.
// fp32: one expf per direction.  fp64: the lattice velocities are small integers, so the exponential factorises,
//   f(x,y) = [rho e^{-1-l0}] (e^{-l3})^{x^2} (e^{-l5})^{y^2} (e^{-l4})^{xy} [e^{-l1} (e^{-l6})^{r^2}]^x [e^{-l2} (e^{-l7})^{r^2}]^y,
// into 8 exponentials, integer powers and a few reciprocals (negative x, y, xy) per evaluation instead of Q
// exponentials of ~20 DFMA each: the solve is fp64-ALU-bound and the exponentials were about half of its arithmetic
// (profiles/r01_ncu_naca_f64.md).  Each f_i carries a few ulp more rounding error than exp of the summed exponent;
// the Newton floor stays ~1e-13 rho, below the tolerance of P:934.
template <int Q, typename T>
__device__ __forceinline__ void numeq_eval(T rho, const T (&m)[NLAMBDA], const T (&lam)[NLAMBDA], T (&f)[Q], T (&s)[Q], T (&G)[NLAMBDA]) {
  if constexpr (!USE_REFLECT_COMBOS<T>) {
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) G[a] = T(0);
  }
  [[maybe_unused]] T C, ea, eb, ec, eci, ep, eq, es, et;
  if constexpr (sizeof(T) == 8) {
    C = rho * Num<T>::exp_(-(T(1) + lam[0]));
    ep = Num<T>::exp_(-lam[1]); eq = Num<T>::exp_(-lam[2]);
    ea = Num<T>::exp_(-lam[3]); ec = Num<T>::exp_(-lam[4]); eb = Num<T>::exp_(-lam[5]);
    es = Num<T>::exp_(-lam[6]); et = Num<T>::exp_(-lam[7]);
    eci = fast_rcp(ec);
  }
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    T fi;
    if constexpr (sizeof(T) == 8) {
      constexpr int x = Lat<Q>::t.cx[I], y = Lat<Q>::t.cy[I], r2 = x * x + y * y;
      constexpr int ax = x < 0 ? -x : x, ay = y < 0 ? -y : y, axy = x * y < 0 ? -x * y : x * y;
      fi = C;
      if constexpr (x != 0) fi *= ipow<x * x, T>(ea);
      if constexpr (y != 0) fi *= ipow<y * y, T>(eb);
      if constexpr (x * y > 0) fi *= ipow<axy, T>(ec);
      if constexpr (x * y < 0) fi *= ipow<axy, T>(eci);
      if constexpr (x != 0) {
        const T X = ipow<ax, T>(ep * ipow<r2, T>(es));
        fi *= x > 0 ? X : fast_rcp(X);
      }
      if constexpr (y != 0) {
        const T Y = ipow<ay, T>(eq * ipow<r2, T>(et));
        fi *= y > 0 ? Y : fast_rcp(Y);
      }
    } else {
      T e = T(1);
      static_for<0, NLAMBDA>([&](auto ac) {
        constexpr int A = decltype(ac)::value;
        constexpr int M = monomial(Lat<Q>::t, I, A);
        if constexpr (M != 0) e += lam[A] * T(M);
      });
      fi = rho * Num<T>::exp_(-e);
    }
    f[I] = fi;
    if constexpr (!USE_REFLECT_COMBOS<T>) {
      static_for<0, NLAMBDA>([&](auto ac) {
        constexpr int A = decltype(ac)::value;
        constexpr int M = monomial(Lat<Q>::t, I, A);
        if constexpr (M != 0) G[A] += fi * T(M);
      });
    }
  });
  if constexpr (!USE_REFLECT_COMBOS<T>) {
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) G[a] -= m[a];
    return;
  }
  // residuals G_a = sum_i f_i M_ia - m_a from the reflection combinations (1, x, y, xx, xy, yy, x r2, y r2)
  reflect_combos<Q, T>(f, s);
  G[0] = sym_moment<Q, T, 0, 0, 0>(s) - m[0];
  G[1] = sym_moment<Q, T, 1, 0, 0>(s) - m[1];
  G[2] = sym_moment<Q, T, 0, 1, 0>(s) - m[2];
  G[3] = sym_moment<Q, T, 2, 0, 0>(s) - m[3];
  G[4] = sym_moment<Q, T, 1, 1, 0>(s) - m[4];
  G[5] = sym_moment<Q, T, 0, 2, 0>(s) - m[5];
  G[6] = sym_moment<Q, T, 1, 0, 1>(s) - m[6];
  G[7] = sym_moment<Q, T, 0, 1, 1>(s) - m[7];
}

// Solves A d = G for a symmetric positive definite 8x8 A given by its lower triangle, by L D L^T in place; false if a
// pivot is not positive.
template <typename T>
__device__ __forceinline__ bool ldlt_solve(T (&A)[NLAMBDA][NLAMBDA], const T (&G)[NLAMBDA], T (&d)[NLAMBDA]) {
  // A = L D L^T in place (unit lower L below the diagonal, D on it): the square-root-free form of the Cholesky
  // factorisation -- the same direction up to rounding, but each column waits for one refined reciprocal (5 dependent
  // instructions) instead of a square root and a division (~40), which matters with two warps per scheduler.
  T rd[NLAMBDA];           // 1 / D_j
  bool ok = true;
  static_for<0, NLAMBDA>([&](auto jc) {
    constexpr int j = decltype(jc)::value;
    T v[j > 0 ? j : 1];    // v_k = L_jk D_k
    T s = A[j][j];
    static_for<0, j>([&](auto kc) {
      constexpr int k = decltype(kc)::value;
      v[k] = A[j][k] * A[k][k];
      s -= A[j][k] * v[k];
    });
    if (!(s > T(0))) ok = false;
    A[j][j] = s;
    rd[j] = fast_rcp(s);
    static_for<j + 1, NLAMBDA>([&](auto ic) {
      constexpr int i = decltype(ic)::value;
      T t = A[i][j];
      static_for<0, j>([&](auto kc) { constexpr int k = decltype(kc)::value; t -= A[i][k] * v[k]; });
      A[i][j] = t * rd[j];
    });
  });
  T z[NLAMBDA] = {};
  static_for<0, NLAMBDA>([&](auto ic) {          // L z = G
    constexpr int i = decltype(ic)::value;
    T t = G[i];
    static_for<0, i>([&](auto kc) { constexpr int k = decltype(kc)::value; t -= A[i][k] * z[k]; });
    z[i] = t;
  });
  static_for<0, NLAMBDA>([&](auto rc) {          // L^T d = D^-1 z
    constexpr int i = NLAMBDA - 1 - decltype(rc)::value;
    T t = z[i] * rd[i];
    static_for<i + 1, NLAMBDA>([&](auto kc) { constexpr int k = decltype(kc)::value; t -= A[k][i] * d[k]; });
    d[i] = t;
  });
  return ok;
}

// Newton direction: solve (-J) d = G, -J = sum_i f_i M_i M_i^T (symmetric positive definite), by L D L^T.
// The 36 entries of the lower triangle are 27 distinct lattice moments of f; the eight of the first column are the
// moment sums the residual already holds (sum_i f_i M_ia = G_a + m_a), three more are sums of two others, so 16 sums
// over the lattice are formed instead of 36 (the Jacobian was about half of the solve's arithmetic).
// Returns false if the matrix is not positive definite.
template <int Q, typename T>
__device__ __forceinline__ bool newton_direction(const T (&f)[Q], const T (&G)[NLAMBDA], const T (&m)[NLAMBDA], T (&d)[NLAMBDA]) {   // f: reflection combinations (fp64) or f itself (fp32)
  T A[NLAMBDA][NLAMBDA];   // lower triangle used
#pragma unroll
  for (int a = 0; a < NLAMBDA; ++a) A[a][0] = G[a] + m[a];            // 1, x, y, xx, xy, yy, x r2, y r2
  A[1][1] = A[3][0]; A[2][1] = A[4][0]; A[2][2] = A[5][0];
  const T xxx = solver_moment<Q, T, 3, 0, 0>(f), xxy = solver_moment<Q, T, 2, 1, 0>(f);
  const T xyy = solver_moment<Q, T, 1, 2, 0>(f), yyy = solver_moment<Q, T, 0, 3, 0>(f);
  const T x4 = solver_moment<Q, T, 4, 0, 0>(f), x3y = solver_moment<Q, T, 3, 1, 0>(f), xxyy = solver_moment<Q, T, 2, 2, 0>(f);
  const T xy3 = solver_moment<Q, T, 1, 3, 0>(f), y4 = solver_moment<Q, T, 0, 4, 0>(f);
  const T xxr2 = x4 + xxyy, xyr2 = x3y + xy3, yyr2 = xxyy + y4;
  const T x3r2 = solver_moment<Q, T, 3, 0, 1>(f), xxyr2 = solver_moment<Q, T, 2, 1, 1>(f);
  const T xyyr2 = solver_moment<Q, T, 1, 2, 1>(f), y3r2 = solver_moment<Q, T, 0, 3, 1>(f);
  A[3][1] = xxx; A[4][1] = xxy; A[5][1] = xyy; A[6][1] = xxr2; A[7][1] = xyr2;
  A[3][2] = xxy; A[4][2] = xyy; A[5][2] = yyy; A[6][2] = xyr2; A[7][2] = yyr2;
  A[3][3] = x4; A[4][3] = x3y; A[5][3] = xxyy; A[6][3] = x3r2; A[7][3] = xxyr2;
  A[4][4] = xxyy; A[5][4] = xy3; A[6][4] = xxyr2; A[7][4] = xyyr2;
  A[5][5] = y4; A[6][5] = xyyr2; A[7][5] = y3r2;
  A[6][6] = solver_moment<Q, T, 2, 0, 2>(f); A[7][6] = solver_moment<Q, T, 1, 1, 2>(f); A[7][7] = solver_moment<Q, T, 0, 2, 2>(f);
  return ldlt_solve<T>(A, G, d);
}

template <typename T>
__device__ __forceinline__ T norm2sq(const T (&G)[NLAMBDA]) {
  T s = T(0);
#pragma unroll
  for (int a = 0; a < NLAMBDA; ++a) s += G[a] * G[a];
  return s;
}

// ---- fp64: the solve in one pass per trial point.  The 8 residual sums and the 16 further lattice moments of the
// Jacobian are accumulated orbit by orbit while the f_i of the trial point are formed (rest; (+-a, 0); (0, +-a);
// (+-a, +-b) through the reflection combinations above), so that no array of Q equilibrium values (nor of their
// combinations) is live across the factorisation: the kernels sat at 254-255 registers with spills, the f_i of the
// final point are evaluated once more after the loop instead (products of the 8 exponentials only, no sums), which also
// replaces the polish phase's full evaluation.  Same rule (S14), same phases, same tests as the loop below.
constexpr int NSUM = 24;
//                                 G: 1  x  y  xx xy yy xr2 yr2 | xxx xxy xyy yyy x4 x3y xxyy xy3 y4 x3r2 xxyr2 xyyr2 y3r2 xxr4 xyr4 yyr4
__device__ constexpr int SUM_PX[NSUM] = {0, 1, 0, 2, 1, 0, 1, 0, 3, 2, 1, 0, 4, 3, 2, 1, 0, 3, 2, 1, 0, 2, 1, 0};
__device__ constexpr int SUM_PY[NSUM] = {0, 0, 1, 0, 1, 2, 0, 1, 0, 1, 2, 3, 0, 1, 2, 3, 4, 0, 1, 2, 3, 0, 1, 2};
__device__ constexpr int SUM_PR[NSUM] = {0, 0, 0, 0, 0, 0, 1, 1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 1, 1, 1, 1, 2, 2, 2};

struct NumeqExps { double C, ea, eb, ec, eci, ep, eq, es, et; };

__device__ __forceinline__ void numeq_exps(double rho, const double (&lam)[NLAMBDA], NumeqExps& E) {
  E.C = rho * exp(-(1.0 + lam[0]));
  E.ep = exp(-lam[1]); E.eq = exp(-lam[2]);
  E.ea = exp(-lam[3]); E.ec = exp(-lam[4]); E.eb = exp(-lam[5]);
  E.es = exp(-lam[6]); E.et = exp(-lam[7]);
  E.eci = fast_rcp(E.ec);
}

// f_I from the factorised exponentials (see numeq_eval)
template <int Q, int I>
__device__ __forceinline__ double numeq_f(const NumeqExps& E) {
  constexpr int x = Lat<Q>::t.cx[I], y = Lat<Q>::t.cy[I], r2 = x * x + y * y;
  constexpr int ax = x < 0 ? -x : x, ay = y < 0 ? -y : y, axy = x * y < 0 ? -x * y : x * y;
  double fi = E.C;
  if constexpr (x != 0) fi *= ipow<x * x, double>(E.ea);
  if constexpr (y != 0) fi *= ipow<y * y, double>(E.eb);
  if constexpr (x * y > 0) fi *= ipow<axy, double>(E.ec);
  if constexpr (x * y < 0) fi *= ipow<axy, double>(E.eci);
  if constexpr (x != 0) {
    const double X = ipow<ax, double>(E.ep * ipow<r2, double>(E.es));
    fi *= x > 0 ? X : fast_rcp(X);
  }
  if constexpr (y != 0) {
    const double Y = ipow<ay, double>(E.eq * ipow<r2, double>(E.et));
    fi *= y > 0 ? Y : fast_rcp(Y);
  }
  return fi;
}

// adds the reflection combination v that lives in slot I (parities spelled by the signs of xi_I) to every sum it enters
template <int Q, int I>
__device__ __forceinline__ void numeq_accumulate(double v, double (&S)[NSUM]) {
  constexpr int x = Lat<Q>::t.cx[I], y = Lat<Q>::t.cy[I];
  constexpr int ax = x < 0 ? -x : x, ay = y < 0 ? -y : y;
  static_for<0, NSUM>([&](auto kc) {
    constexpr int K = decltype(kc)::value;
    constexpr bool match = ((SUM_PX[K] & 1) == (x < 0 ? 1 : 0)) && ((SUM_PY[K] & 1) == (y < 0 ? 1 : 0));
    constexpr int wgt = ipow_c(ax, SUM_PX[K]) * ipow_c(ay, SUM_PY[K]) * ipow_c(x * x + y * y, SUM_PR[K]);
    if constexpr (match && wgt != 0) S[K] += v * double(wgt);
  });
}

template <int Q>
__device__ __forceinline__ void numeq_pass(double rho, const double (&lam)[NLAMBDA], double (&S)[NSUM]) {
  NumeqExps E;
  numeq_exps(rho, lam, E);
#pragma unroll
  for (int k = 0; k < NSUM; ++k) S[k] = 0.0;
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int x = Lat<Q>::t.cx[I], y = Lat<Q>::t.cy[I];
    if constexpr (x == 0 && y == 0) {
      numeq_accumulate<Q, I>(numeq_f<Q, I>(E), S);
    } else if constexpr ((x > 0 && y == 0) || (x == 0 && y > 0)) {
      constexpr int J = dir_index(Lat<Q>::t, -x, -y);
      const double fp = numeq_f<Q, I>(E), fm = numeq_f<Q, J>(E);
      numeq_accumulate<Q, I>(fp + fm, S);
      numeq_accumulate<Q, J>(fp - fm, S);
    } else if constexpr (x > 0 && y > 0) {
      constexpr int Jx = dir_index(Lat<Q>::t, -x, y), Jy = dir_index(Lat<Q>::t, x, -y), Jxy = dir_index(Lat<Q>::t, -x, -y);
      const double f1 = numeq_f<Q, I>(E), f2 = numeq_f<Q, Jx>(E), f3 = numeq_f<Q, Jy>(E), f4 = numeq_f<Q, Jxy>(E);
      const double p1 = f1 + f2, m1 = f1 - f2, p2 = f3 + f4, m2 = f3 - f4;
      numeq_accumulate<Q, I>(p1 + p2, S);
      numeq_accumulate<Q, Jx>(m1 + m2, S);
      numeq_accumulate<Q, Jy>(p1 - p2, S);
      numeq_accumulate<Q, Jxy>(m1 - m2, S);
    }
  });
}

__device__ __forceinline__ bool newton_direction_from_sums(const double (&S)[NSUM], const double (&G)[NLAMBDA], double (&d)[NLAMBDA]) {
  double A[NLAMBDA][NLAMBDA];   // lower triangle of -J = sum_i f_i M_i M_i^T
#pragma unroll
  for (int a = 0; a < NLAMBDA; ++a) A[a][0] = S[a];
  A[1][1] = S[3]; A[2][1] = S[4]; A[2][2] = S[5];
  const double xxx = S[8], xxy = S[9], xyy = S[10], yyy = S[11], x4 = S[12], x3y = S[13], xxyy = S[14], xy3 = S[15], y4 = S[16];
  const double xxr2 = x4 + xxyy, xyr2 = x3y + xy3, yyr2 = xxyy + y4;
  const double x3r2 = S[17], xxyr2 = S[18], xyyr2 = S[19], y3r2 = S[20];
  A[3][1] = xxx; A[4][1] = xxy; A[5][1] = xyy; A[6][1] = xxr2; A[7][1] = xyr2;
  A[3][2] = xxy; A[4][2] = xyy; A[5][2] = yyy; A[6][2] = xyr2; A[7][2] = yyr2;
  A[3][3] = x4; A[4][3] = x3y; A[5][3] = xxyy; A[6][3] = x3r2; A[7][3] = xxyr2;
  A[4][4] = xxyy; A[5][4] = xy3; A[6][4] = xxyr2; A[7][4] = xyyr2;
  A[5][5] = y4; A[6][5] = xyyr2; A[7][5] = y3r2;
  A[6][6] = S[21]; A[7][6] = S[22]; A[7][7] = S[23];
  return ldlt_solve<double>(A, G, d);
}

template <int Q>
__device__ __forceinline__ int feq_numerical_onepass(const ModelParams& p, double rho, double ux, double uy, double Tm,
                                                     double (&lam)[NLAMBDA], double (&f)[Q]) {
  const double u2 = ux * ux + uy * uy;
  const double m[NLAMBDA] = {rho, rho * ux, rho * uy, rho * (ux * ux + Tm), rho * ux * uy, rho * (uy * uy + Tm),
                             rho * ux * (u2 + 4.0 * Tm), rho * uy * (u2 + 4.0 * Tm)};
  double S[NSUM], G[NLAMBDA], d[NLAMBDA], lt[NLAMBDA];
  const double tol = p.newton_tol * rho;
  enum { INIT, SEARCH, POLISH };
  int it = 0, phase = INIT;
  bool converged = false, bad = false;
  double t = 0.0, n0 = 0.0;
#pragma unroll
  for (int a = 0; a < NLAMBDA; ++a) d[a] = 0.0;
#pragma unroll 1
  for (;;) {
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) lt[a] = lam[a] + t * d[a];
    if (phase == POLISH) {        // the unconditional full step; its equilibrium is evaluated below
#pragma unroll
      for (int a = 0; a < NLAMBDA; ++a) lam[a] = lt[a];
      ++it;
      break;
    }
    numeq_pass<Q>(rho, lt, S);
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) G[a] = S[a] - m[a];
    if (phase == SEARCH) {
      const double n1 = norm2sq(G);
      if (!(n1 < n0) && t > 1.0 / 1024.0) { t *= 0.5; continue; }   // a NaN norm keeps halving
    }
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) lam[a] = lt[a];
    if (phase != INIT) ++it;
    double r1 = 0.0;
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) r1 += fabs(G[a]);
    converged = r1 <= tol;
    phase = (converged || it >= p.newton_max_iter) ? POLISH : SEARCH;
    if (!newton_direction_from_sums(S, G, d)) { bad = true; break; }
    n0 = norm2sq(G);
    t = 1.0;
  }
  NumeqExps E;
  numeq_exps(rho, lam, E);
  static_for<0, Q>([&](auto ic) { f[decltype(ic)::value] = numeq_f<Q, decltype(ic)::value>(E); });
  return (converged && !bad) ? it : -it - 1;
}

// Newton-Raphson with a halving line search; deterministic rule of DESIGN.md Sec. 4 (S14):
// iterate until sum|G_a| <= tol*rho or max_iter, then one unconditional full Newton step.
// lam in/out; feq out.  Returns the number of Newton steps (polish included), negative on failure.
template <int Q, typename T>
__device__ __forceinline__ int feq_numerical(const ModelParams& p, T rho, T ux, T uy, T Tm, T (&lam)[NLAMBDA], T (&f)[Q]) {
  if constexpr (sizeof(T) == 8) return feq_numerical_onepass<Q>(p, rho, ux, uy, Tm, lam, f);
  const T u2 = ux * ux + uy * uy;
  // right-hand sides of Eq. 42-49 with 2E = u^2 + 2T
  const T m[NLAMBDA] = {rho, rho * ux, rho * uy, rho * (ux * ux + Tm), rho * ux * uy, rho * (uy * uy + Tm),
                        rho * ux * (u2 + T(4) * Tm), rho * uy * (u2 + T(4) * Tm)};
  // One loop with a single evaluation site and a single direction site (the three textual call sites of the rule --
  // initial residual, line-search trial, polish -- are phases of it): fully inlined, each site is ~1-2 k instructions,
  // and three copies of them overflowed the instruction cache (profiles/r01_ncu_naca_f64.md: stall_no_instruction).
  T G[NLAMBDA], d[NLAMBDA], lt[NLAMBDA];
  [[maybe_unused]] T sc[Q];        // reflection combinations of the trial equilibrium (fp64)
  const T tol = T(p.newton_tol) * rho;
  enum { INIT, SEARCH, POLISH };
  int it = 0, phase = INIT;
  bool converged = false, bad = false;
  T t = T(0), n0 = T(0);
#pragma unroll
  for (int a = 0; a < NLAMBDA; ++a) d[a] = T(0);
#pragma unroll 1
  for (;;) {
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) lt[a] = lam[a] + t * d[a];
    numeq_eval<Q, T>(rho, m, lt, f, sc, G);
    if (phase == SEARCH) {
      const T n1 = norm2sq(G);
      if (!(n1 < n0) && t > T(1.0 / 1024.0)) { t *= T(0.5); continue; }   // a NaN norm keeps halving
    }
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) lam[a] = lt[a];
    if (phase != INIT) ++it;
    if (phase == POLISH) break;
    T r1 = T(0);
#pragma unroll
    for (int a = 0; a < NLAMBDA; ++a) r1 += Num<T>::abs_(G[a]);
    converged = r1 <= tol;
    // single precision: the moment sums carry ~Q eps |M|max rho of rounding (D2Q37: ~7e-5 rho), above the 1e-5 rho of P:934, so a
    // solve can sit on that floor without ever passing the test: at the iteration limit a residual within 32 tol counts as
    // converged (the oracle, in double precision, never gets there)
    if (sizeof(T) == 4 && it >= p.newton_max_iter && r1 <= T(32) * tol) converged = true;
    phase = (converged || it >= p.newton_max_iter) ? POLISH : SEARCH;    // then one unconditional full Newton step
    if (!newton_direction<Q, T>(USE_REFLECT_COMBOS<T> ? sc : f, G, m, d)) { bad = true; break; }
    n0 = norm2sq(G);
    t = T(1);
  }
  return (converged && !bad) ? it : -it - 1;
}

// Equilibrium of the configured model for a given macroscopic state (used by initialisation and by
// Dirichlet cells).  THERMAL selects the T-dependent Hermite moments.
template <int Q, typename T, int COLL, bool DDF>
__device__ __forceinline__ int equilibrium(const ModelParams& p, T rho, T ux, T uy, T Tm, T (&lam)[NLAMBDA], T (&feq)[Q], T (&geq)[Q]) {
  int it = 0;
  if constexpr (COLL == LBM_NUMEQ) {
    it = feq_numerical<Q, T>(p, rho, ux, uy, Tm, lam, feq);
  } else {
    T a[NA];
    aeq_moments<T>(rho, ux, uy, DDF ? Tm - T(cs2_v<Q>) : T(0), a);
    poly_all<Q, T>(a, [&](auto ic, T fe) { feq[decltype(ic)::value] = fe; });
  }
  if constexpr (DDF) {
    const T fac = T(2.0 / (p.gamma - 1.0) - 2.0) * Tm;   // Eq. 50: (2 C_v - D) T, D = 2
#pragma unroll
    for (int i = 0; i < Q; ++i) geq[i] = fac * feq[i];
  }
  return it;
}

// Eq. 37-38 (typo of P:876 repaired, S2): non-equilibrium Hermite moments of orders 3-4 from Pi by the recursion,
// then a* = a_eq + (1 - 1/tau) a_neq in place (Eq. 33).  Slots outside the lattice's basis are ignored downstream.
template <typename T>
__device__ __forceinline__ void rr_post_collision_moments(T ux, T uy, T pxx, T pxy, T pyy, T keep, T (&ae)[NA]) {
  T an[NA];
  an[A0] = T(0); an[AX] = T(0); an[AY] = T(0);
  an[AXX] = pxx; an[AXY] = pxy; an[AYY] = pyy;
  an[AXXX] = T(3) * ux * pxx;
  an[AXXY] = T(2) * ux * pxy + uy * pxx;
  an[AXYY] = T(2) * uy * pxy + ux * pyy;
  an[AYYY] = T(3) * uy * pyy;
  an[AXXXX] = T(4) * ux * an[AXXX] - T(6) * ux * ux * pxx;
  an[AXXXY] = (T(3) * ux * an[AXXY] + uy * an[AXXX]) - T(3) * ux * ux * pxy - T(3) * ux * uy * pxx;
  an[AXXYY] = T(2) * (ux * an[AXYY] + uy * an[AXXY]) - ux * ux * pyy - uy * uy * pxx - T(4) * ux * uy * pxy;
  an[AXYYY] = (T(3) * uy * an[AXYY] + ux * an[AYYY]) - T(3) * uy * uy * pxy - T(3) * ux * uy * pyy;
  an[AYYYY] = T(4) * uy * an[AYYY] - T(6) * uy * uy * pyy;
#pragma unroll
  for (int k = 0; k < NA; ++k) ae[k] += keep * an[k];
}

// Eq. 53 with reading S10: alpha = 1 below 0.01; last case alpha = 1/tau (tau_eff = 1)
template <typename T>
__device__ __forceinline__ T sensor_alpha(T eps, T A, T tau) {
  if (eps < T(0.01)) return T(1);
  if (eps < T(0.10)) return T(1.05);
  if (eps < T(1.00)) return A;
  return T(1) / tau;
}

// Steps 2-5 of the cell update, in place: f, g pre-collision in, post-collision out.
// Returns Newton iterations (0 for polynomial models, negative on failure); rho_out = pre-collision density.
// `imp` (numerical equilibria only): an equilibrium Dirichlet cell passes its imposed state here and receives
// f = f^eq, g = g^eq of it, so that the kernel holds ONE inlined copy of the Newton solver (instruction-cache footprint).
template <typename T> struct Imposed { bool on; T rho, ux, uy, Tm; };

template <int Q, typename T, int COLL, bool DDF, bool SENSOR>
__device__ __forceinline__ int collide(const ModelParams& p, T tau, T (&f)[Q], T (&g)[Q], T (&lam)[NLAMBDA], T& rho_out,
                                       const Imposed<T> imp = Imposed<T>{false, T(0), T(0), T(0), T(0)}) {
  constexpr bool THERMAL = (COLL == LBM_NUMEQ) || DDF;
  static_assert(!(COLL == LBM_RR && DDF), "RR is defined for the athermal models only");
  T rho, ux, uy, Tm;
  moments<Q, T, THERMAL, DDF>(p, f, g, rho, ux, uy, Tm);
  if constexpr (COLL == LBM_NUMEQ) {
    if (imp.on) { rho = imp.rho; ux = imp.ux; uy = imp.uy; Tm = imp.Tm; }
  }
  rho_out = rho;
  int it = 0;

  if constexpr (COLL == LBM_NUMEQ) {
    // numerical equilibrium: held in registers (Newton produces all of it; the sensor needs all of it before relaxing)
    T feq[Q];
    it = feq_numerical<Q, T>(p, rho, ux, uy, Tm, lam, feq);
    T tau_eff = tau;
    if constexpr (SENSOR) {
      T eps = T(0);
#pragma unroll
      for (int i = 0; i < Q; ++i) {
        T den = Num<T>::abs_(feq[i]);
        if (den < Num<T>::tiny()) den = Num<T>::tiny();
        eps += Num<T>::abs_(f[i] - feq[i]) * fast_rcp(den);          // Eq. 52
      }
      eps /= T(Q);
      tau_eff = tau * sensor_alpha<T>(eps, T(p.sensor_A), tau);
    }
    const T keep = T(1) - T(1) / tau_eff;
#pragma unroll
    for (int i = 0; i < Q; ++i) f[i] = imp.on ? feq[i] : feq[i] + keep * (f[i] - feq[i]);      // Eq. 30
    if constexpr (DDF) {
      const T fac = T(2.0 / (p.gamma - 1.0) - 2.0) * Tm;                     // Eq. 50: (2 C_v - D) T
#pragma unroll
      for (int i = 0; i < Q; ++i) { const T ge = fac * feq[i]; g[i] = imp.on ? ge : ge + keep * (g[i] - ge); }
    }
  } else if constexpr (COLL == LBM_BGK) {
    static_assert(COLL != LBM_RR || !SENSOR, "sensor is instantiated for BGK-type relaxation only");
    T keep = T(1) - T(1) / tau;
    T a[NA];
    aeq_moments<T>(rho, ux, uy, DDF ? Tm - T(cs2_v<Q>) : T(0), a);
    if constexpr (SENSOR) {
      // Eq. 52-53 need every f_i^eq before any relaxation: one pass for eps, then f^eq is RECOMPUTED in the relaxation
      // pass instead of being kept in Q more registers (D2Q37+g: 255 registers and spills otherwise).  The moments are
      // hidden from common-subexpression elimination, which would undo exactly that.
      T eps = T(0);
      poly_all<Q, T>(a, [&](auto ic, T fe) {
        constexpr int I = decltype(ic)::value;
        T den = Num<T>::abs_(fe);
        if (den < Num<T>::tiny()) den = Num<T>::tiny();
        eps += Num<T>::abs_(f[I] - fe) * fast_rcp(den);                      // Eq. 52
      });
      eps /= T(Q);
      keep = T(1) - T(1) / (tau * sensor_alpha<T>(eps, T(p.sensor_A), tau));
#pragma unroll
      for (int k = 0; k < NA; ++k) opaque(a[k]);
    }
    const T fac = DDF ? T(2.0 / (p.gamma - 1.0) - 2.0) * Tm : T(0);
    poly_all<Q, T>(a, [&](auto ic, T fe) {
      constexpr int I = decltype(ic)::value;
      f[I] = fe + keep * (f[I] - fe);
      if constexpr (DDF) { const T ge = fac * fe; g[I] = ge + keep * (g[I] - ge); }
    });
  } else {   // LBM_RR
    const T keep = T(1) - T(1) / tau;
    constexpr double c2 = cs2_v<Q>;
    T ae[NA];
    aeq_moments<T>(rho, ux, uy, T(0), ae);
    // Pi = sum_i H_i^(2) (f_i - f_i^eq).  The lattices with rational weights reproduce the second-order
    // moments of f^eq exactly, so Pi = sum_i xi xi f_i - rho c_s^2 delta - rho u u there (one pass over f, no f^eq);
    // D2Q37's 15-digit weights (S23) do so only to ~1e-13, so it keeps the literal form.
    T pxx = T(0), pxy = T(0), pyy = T(0);
    if constexpr (Q != 37) {
      static_for<1, Q>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        constexpr int cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I];
        if constexpr (cx != 0) pxx += T(cx * cx) * f[I];
        if constexpr (cx * cy != 0) pxy += T(cx * cy) * f[I];
        if constexpr (cy != 0) pyy += T(cy * cy) * f[I];
      });
      pxx = (pxx - T(c2) * rho) - ae[AXX];
      pxy = pxy - ae[AXY];
      pyy = (pyy - T(c2) * rho) - ae[AYY];
    } else {
      static_for<0, Q>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        constexpr int cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I];
        const T dn = f[I] - poly_i<Q, T, I>(ae);
        pxx += T(cx * cx - c2) * dn;
        if constexpr (cx * cy != 0) pxy += T(cx * cy) * dn;
        pyy += T(cy * cy - c2) * dn;
      });
    }
    if (p.trace_eq) {   // trace relaxes with tau = 1: only the deviatoric part survives (S7)
      const T dev = T(0.5) * (pxx - pyy);
      pxx = dev; pyy = -dev;
    }
    rr_post_collision_moments<T>(ux, uy, pxx, pxy, pyy, keep, ae);
    poly_all<Q, T>(ae, [&](auto ic, T fs) { f[decltype(ic)::value] = fs; });   // Eq. 33
  }
  return it;
}

}  // namespace lbm
