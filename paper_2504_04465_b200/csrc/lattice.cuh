// lattice.cuh -- compile-time lattice tables and Hermite coefficients of the CUDA path.
// Table 4, Table 5, Eq. 34-35.  Everything here is evaluated by
// the compiler: the kernels see immediates only (no constant-memory tables, no indexed loads).
#pragma once
#include <type_traits>

namespace lbm {

constexpr int QMAX = 37;
constexpr int NLAMBDA = 8;

struct LatTab {
  int Q = 0, W = 0;
  double cs2 = 0.0;
  int cx[QMAX] = {}, cy[QMAX] = {}, opp[QMAX] = {};
  double w[QMAX] = {};
  // basis of Table 5: third order full (xxx, yyy) / mixed (xxy, xyy); fourth order xxyy / full
  bool h3_full = false, h3_mixed = false, h4_xxyy = false, h4_full = false;
};

__host__ __device__ constexpr void lat_put_group(LatTab& L, int a, int b, double w) {
  // canonical order inside a group: counter-clockwise from the +x axis
  int n = L.Q;
  if (a == 0) {
    L.cx[n] = 0; L.cy[n] = 0; L.w[n] = w; n += 1;
  } else if (b == 0) {
    const int X[4] = {a, 0, -a, 0}, Y[4] = {0, a, 0, -a};
    for (int k = 0; k < 4; ++k) { L.cx[n] = X[k]; L.cy[n] = Y[k]; L.w[n] = w; ++n; }
  } else if (a == b) {
    const int X[4] = {a, -a, -a, a}, Y[4] = {a, a, -a, -a};
    for (int k = 0; k < 4; ++k) { L.cx[n] = X[k]; L.cy[n] = Y[k]; L.w[n] = w; ++n; }
  } else {
    const int X[8] = {a, b, -b, -a, -a, -b, b, a}, Y[8] = {b, a, a, b, -b, -a, -a, -b};
    for (int k = 0; k < 8; ++k) { L.cx[n] = X[k]; L.cy[n] = Y[k]; L.w[n] = w; ++n; }
  }
  L.Q = n;
  const int r = a > b ? a : b;
  if (r > L.W) L.W = r;
}

__host__ __device__ constexpr LatTab make_lat(int Q) {
  LatTab L;
  if (Q == 9) {            // D2Q9: c_s^2 = 1/3, partial 4th-order basis
    lat_put_group(L, 0, 0, 4.0 / 9.0); lat_put_group(L, 1, 0, 1.0 / 9.0); lat_put_group(L, 1, 1, 1.0 / 36.0);
    L.cs2 = 1.0 / 3.0; L.h3_mixed = true; L.h4_xxyy = true;
  } else if (Q == 13) {    // D2Q13: c_s^2 = 1/2, full 3rd order
    lat_put_group(L, 0, 0, 3.0 / 8.0); lat_put_group(L, 1, 0, 1.0 / 12.0); lat_put_group(L, 1, 1, 1.0 / 16.0);
    lat_put_group(L, 2, 0, 1.0 / 96.0);
    L.cs2 = 0.5; L.h3_full = true; L.h3_mixed = true;
  } else if (Q == 21) {    // D2Q21: c_s^2 = 2/3, full 3rd order
    lat_put_group(L, 0, 0, 91.0 / 324.0); lat_put_group(L, 1, 0, 1.0 / 12.0); lat_put_group(L, 1, 1, 2.0 / 27.0);
    lat_put_group(L, 2, 0, 7.0 / 360.0); lat_put_group(L, 2, 2, 1.0 / 432.0); lat_put_group(L, 3, 0, 1.0 / 1620.0);
    L.cs2 = 2.0 / 3.0; L.h3_full = true; L.h3_mixed = true;
  } else if (Q == 37) {    // D2Q37: 15-digit decimals of Table 4 verbatim (reading S23), full 4th order
    lat_put_group(L, 0, 0, 0.233150669132352); lat_put_group(L, 1, 0, 0.107306091542219);
    lat_put_group(L, 1, 1, 0.057667859888794); lat_put_group(L, 2, 0, 0.014208216158450);
    lat_put_group(L, 2, 1, 0.005353049000513); lat_put_group(L, 2, 2, 0.001011937592673);
    lat_put_group(L, 3, 0, 0.000245301027757); lat_put_group(L, 3, 1, 0.000283414252994);
    L.cs2 = 0.697953322019683; L.h3_full = true; L.h3_mixed = true; L.h4_xxyy = true; L.h4_full = true;
  }
  for (int i = 0; i < L.Q; ++i)
    for (int j = 0; j < L.Q; ++j)
      if (L.cx[j] == -L.cx[i] && L.cy[j] == -L.cy[i]) L.opp[i] = j;
  return L;
}

template <int Q>
struct Lat {
  static constexpr LatTab t = make_lat(Q);
  static_assert(t.Q == Q, "unknown lattice");
};

template <int Q> constexpr double cs2_v = make_lat(Q).cs2;   // scalar copies are usable in device code

// Hermite moment slots: 0 | x y | xx xy yy | xxx xxy xyy yyy | xxxx xxxy xxyy xyyy yyyy
enum { A0 = 0, AX, AY, AXX, AXY, AYY, AXXX, AXXY, AXYY, AYYY, AXXXX, AXXXY, AXXYY, AXYYY, AYYYY, NA };

// Coefficient of Hermite moment slot k in f_i of Eq. 33/34:  w_i * mult_k * H_k(xi_i) / (n! c_s^{2n}),
// mult = multiplicity of the component in the full contraction (xy 2, xxy/xyy 3, xxxy/xyyy 4, xxyy 6);
// zero for slots outside the lattice's basis (Table 5).
__host__ __device__ constexpr double hermite_coef(const LatTab& L, int i, int k) {
  const double x = L.cx[i], y = L.cy[i], c2 = L.cs2, c4 = c2 * c2, c6 = c4 * c2, c8 = c4 * c4;
  double h = 0.0;
  switch (k) {
    case A0: h = 1.0; break;
    case AX: h = x / c2; break;
    case AY: h = y / c2; break;
    case AXX: h = (x * x - c2) / (2.0 * c4); break;
    case AXY: h = 2.0 * (x * y) / (2.0 * c4); break;
    case AYY: h = (y * y - c2) / (2.0 * c4); break;
    case AXXX: h = L.h3_full ? (x * x - 3.0 * c2) * x / (6.0 * c6) : 0.0; break;
    case AYYY: h = L.h3_full ? (y * y - 3.0 * c2) * y / (6.0 * c6) : 0.0; break;
    case AXXY: h = L.h3_mixed ? 3.0 * (x * x - c2) * y / (6.0 * c6) : 0.0; break;
    case AXYY: h = L.h3_mixed ? 3.0 * (y * y - c2) * x / (6.0 * c6) : 0.0; break;
    case AXXXX: h = L.h4_full ? (x * x * x * x - 6.0 * c2 * x * x + 3.0 * c4) / (24.0 * c8) : 0.0; break;
    case AYYYY: h = L.h4_full ? (y * y * y * y - 6.0 * c2 * y * y + 3.0 * c4) / (24.0 * c8) : 0.0; break;
    case AXXXY: h = L.h4_full ? 4.0 * (x * x - 3.0 * c2) * x * y / (24.0 * c8) : 0.0; break;
    case AXYYY: h = L.h4_full ? 4.0 * (y * y - 3.0 * c2) * y * x / (24.0 * c8) : 0.0; break;
    case AXXYY: h = L.h4_xxyy ? 6.0 * (x * x - c2) * (y * y - c2) / (24.0 * c8) : 0.0; break;
    default: break;
  }
  return L.w[i] * h;
}

// Monomials paired with the eight multipliers of the numerical equilibrium (Eq. 42-49):
// 1, x, y, xx, xy, yy, x(xx+yy), y(xx+yy)
__host__ __device__ constexpr int monomial(const LatTab& L, int i, int a) {
  const int x = L.cx[i], y = L.cy[i], r2 = x * x + y * y;
  switch (a) {
    case 0: return 1;
    case 1: return x;
    case 2: return y;
    case 3: return x * x;
    case 4: return x * y;
    case 5: return y * y;
    case 6: return x * r2;
    default: return y * r2;
  }
}

// compile-time loop: f(std::integral_constant<int, I>{}) for I = B .. E-1
template <int B, int E, class F>
__device__ __forceinline__ void static_for(F&& f) {
  if constexpr (B < E) {
    f(std::integral_constant<int, B>{});
    static_for<B + 1, E>(f);
  }
}

}  // namespace lbm
