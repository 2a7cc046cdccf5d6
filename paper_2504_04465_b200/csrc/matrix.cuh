// matrix.cuh -- "matrix-like" uniform path: Cartesian-index addressing and AA-pattern in-place
// streaming for single-level boxes, the paper's Eq. 14 roofline point (2 Q s bytes per update, no list) and
// its first "future work" item (one population copy instead of two).
//
// One array A[Q][ny * nx] (row-major, x fastest) holds the state in one of two layouts that alternate with the steps
// (Bailey et al.'s AA pattern; S_i(x) = the canonical post-collision state of DESIGN.md Sec. 2):
//   P0:  A[i][x + xi_i] = S_i(x): slot i of a cell holds f_i(x, t+1), the value it collides with next;
//   P1:  A[opp(i)][x] = S_i(x);
//   in both, where x + xi_i lies behind a wall side: A[opp(i)][x] = S_i(x) + Ladd's term of direction opp(i) with
//   rho_w = sum_k S_k(x) -- exactly what direction opp(i) of the same cell pulls through that wall
//   in the next step.  The term is folded in by the thread that owns the whole state of x when it writes it (a cell's
//   slots are overwritten by its neighbours during an odd step, so rho_w cannot be formed at reading time).
// even step (P0 -> P1): read slot i of the own cell, collide, write slot opp(i) of the own cell -- purely local;
// odd step  (P1 -> P0): read slot opp(i) of x - xi_i, collide, write slot i of x + xi_i -- every thread reads and
//                       writes the same set of addresses, so the update is in place without a second buffer.
// Sides are periodic, bounce-back walls or velocity bounce-back walls (the lid of the cavity), resolved by
// coordinate arithmetic with the builder's corner rule (the y side decides where both are left).
// Weakly compressible models (BGK / RR polynomial), all four lattices, fp64 / fp32; no solids, no refinement.
#pragma once
#include "sweep.cuh"

namespace lbm {

struct MatrixArgs {
  int nx, ny, n;
  long long ps;             // plane stride of A (elements)
  void* A;
  double tau;
  int* status;
  int parity;               // layout of A on entry: 0 = P0, 1 = P1 (I/O kernels)
  const int* pos;           // storage index (Z-curve order of the ABI) -> row-major index iy * nx + ix (I/O kernels)
  const int* cells;         // probe list or null (macroscopic)
  const double* rho; const double* ux; const double* uy;      // init: per storage cell
  double* o_rho; double* o_ux; double* o_uy; double* o_T;     // macroscopic: per output slot
  double* pops;             // export / import: [storage cell][Q]
};

// Row-major index of (x + DX, y + DY) after periodic wrap, or -1 - side if the target lies behind a non-periodic side.
template <int DX, int DY>
__device__ __forceinline__ int matrix_target(const MatrixArgs& a, const ModelParams& p, int x, int y) {
  int tx = x + DX, ty = y + DY;
  if constexpr (DY != 0) {
    if (ty < 0 || ty >= a.ny) {
      if (p.bc_kind[2] != LBM_BC_PERIODIC) return -1 - (ty < 0 ? 2 : 3);
      ty += ty < 0 ? a.ny : -a.ny;
    }
  }
  if constexpr (DX != 0) {
    if (tx < 0 || tx >= a.nx) {
      if (p.bc_kind[0] != LBM_BC_PERIODIC) return -1 - (tx < 0 ? 0 : 1);
      tx += tx < 0 ? a.nx : -a.nx;
    }
  }
  return ty * a.nx + tx;
}

// Ladd's term of direction I pulled through a velocity-bounce-back side: 2 w_i rho_w (xi_i . u_w) / c_s^2 (S11); zero for
// a resting wall
template <int Q, typename T, int I>
__device__ __forceinline__ T matrix_vbb(const ModelParams& p, int side, T rho_w) {
  if (p.bc_kind[side] == LBM_BC_WALL) return T(0);
  constexpr int cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I];
  constexpr double w2 = 2.0 * Lat<Q>::t.w[I];
  const T xu = T(cx) * T(p.bc_ux[side]) + T(cy) * T(p.bc_uy[side]);
  return T(w2) * rho_w * xu / T(cs2_v<Q>);
}

// Cells per thread along x: two where a cell holds <= 104 bytes of populations, as in the brick path (even steps: 128-bit
// accesses in fp64, 64-bit in fp32; odd steps: two independent shifted accesses in flight per direction).  Four cells per
// thread in fp32 was measured slower (uniform 4096^2 D2Q9: 70.3 against 86.2 GLUPS: the grid shrinks and the odd step's
// scalar accesses pile up in the LSU).
template <int Q, typename T> constexpr int MATRIX_CPT = (Q * (int)sizeof(T) <= 104) ? 2 : 1;

// One step.  ODD = layout on entry is P1.  CPT consecutive cells of a row per thread (nx must be a multiple of CPT).
template <int Q, typename T, int COLL, bool ODD, int CPT>
__global__ void __launch_bounds__(128) matrix_step_kernel(const MatrixArgs a, const ModelParams p) {
  const int x0 = ((int)blockIdx.x * 128 + (int)threadIdx.x) * CPT, y = (int)blockIdx.y;
  if (x0 >= a.nx) return;
  T* __restrict__ A = (T*)a.A;
  const long long ps = a.ps;
  const int c0 = y * a.nx + x0;
  constexpr int W = Lat<Q>::t.W;
  T f[CPT][Q], g[Q], lam[NLAMBDA];
  // cells at least W away from every side address their neighbours by a constant offset, no side tests
  const bool interior = y >= W && y < a.ny - W && x0 >= W && x0 + CPT - 1 < a.nx - W;
  if constexpr (!ODD) {
#pragma unroll
    for (int i = 0; i < Q; ++i) {
      const Vec<T, CPT> v = *reinterpret_cast<const Vec<T, CPT>*>(A + i * ps + c0);
#pragma unroll
      for (int j = 0; j < CPT; ++j) f[j][i] = v.v[j];
    }
  } else if (interior) {
    static_for<0, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      constexpr int O = Lat<Q>::t.opp[I], cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I];
      const T* src = A + O * ps + (c0 - cy * a.nx - cx);
#pragma unroll
      for (int j = 0; j < CPT; ++j) f[j][I] = src[j];
    });
  } else {
#pragma unroll
    for (int j = 0; j < CPT; ++j) {
      const int x = x0 + j, c = c0 + j;
      static_for<0, Q>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        constexpr int O = Lat<Q>::t.opp[I];
        const int t = matrix_target<-Lat<Q>::t.cx[I], -Lat<Q>::t.cy[I]>(a, p, x, y);
        // behind a wall: the cell's own slot I = S_opp(I) + Ladd's term of direction I, folded in when it was written
        f[j][I] = t >= 0 ? A[O * ps + t] : A[I * ps + c];
      });
    }
  }
#pragma unroll
  for (int j = 0; j < CPT; ++j) {
    T rho;
    collide<Q, T, COLL, false, false>(p, T(a.tau), f[j], g, lam, rho);
    if (!(rho > T(0)) || !isfinite(rho)) atomicOr(a.status, FLAG_UNSTABLE);
  }
  if constexpr (!ODD) {
    if (!interior) {
#pragma unroll
      for (int j = 0; j < CPT; ++j) {
        T rho_n = T(0);
#pragma unroll
        for (int i = 0; i < Q; ++i) rho_n += f[j][i];          // sum_k S_k of the new state: rho_w of the next pull (S11)
        static_for<1, Q>([&](auto ic) {
          constexpr int I = decltype(ic)::value;
          constexpr int O = Lat<Q>::t.opp[I];
          const int t = matrix_target<Lat<Q>::t.cx[I], Lat<Q>::t.cy[I]>(a, p, x0 + j, y);
          if (t < 0) f[j][I] += matrix_vbb<Q, T, O>(p, -1 - t, rho_n);
        });
      }
    }
    static_for<0, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value, O = Lat<Q>::t.opp[I];
      Vec<T, CPT> v;
#pragma unroll
      for (int j = 0; j < CPT; ++j) v.v[j] = f[j][I];
      *reinterpret_cast<Vec<T, CPT>*>(A + O * ps + c0) = v;
    });
  } else if (interior) {
    static_for<0, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      constexpr int cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I];
      T* dst = A + I * ps + (c0 + cy * a.nx + cx);
#pragma unroll
      for (int j = 0; j < CPT; ++j) dst[j] = f[j][I];
    });
  } else {
#pragma unroll
    for (int j = 0; j < CPT; ++j) {
      const int x = x0 + j, c = c0 + j;
      T rho_n = T(0);
#pragma unroll
      for (int i = 0; i < Q; ++i) rho_n += f[j][i];          // sum_k S_k of the new state: rho_w of the next pull (S11)
      static_for<0, Q>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        constexpr int O = Lat<Q>::t.opp[I];
        const int t = matrix_target<Lat<Q>::t.cx[I], Lat<Q>::t.cy[I]>(a, p, x, y);
        if (t >= 0) A[I * ps + t] = f[j][I];
        else A[O * ps + c] = f[j][I] + matrix_vbb<Q, T, O>(p, -1 - t, rho_n);     // what direction opp(I) pulls next step
      });
    }
  }
}

// The canonical state S_i of the cell at (x, y) out of either layout.  Behind a wall the slot holds S_i + Ladd's term with
// rho_w = sum_k S_k, which is taken out again: the stored values of the cell sum to rho_w (1 + sum over the wall links of
// the term's coefficient).
template <int Q, typename T>
__device__ __forceinline__ void matrix_load_state(const MatrixArgs& a, const ModelParams& p, int x, int y, T (&S)[Q]) {
  const T* __restrict__ A = (const T*)a.A;
  const long long ps = a.ps;
  const int c = y * a.nx + x;
  T sum = T(0), coef = T(0);
  bool wall = false;
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int O = Lat<Q>::t.opp[I];
    const int t = matrix_target<Lat<Q>::t.cx[I], Lat<Q>::t.cy[I]>(a, p, x, y);
    S[I] = (t >= 0 && a.parity == 0) ? A[I * ps + t] : A[O * ps + c];
    sum += S[I];
    if (t < 0) { coef += matrix_vbb<Q, T, O>(p, -1 - t, T(1)); wall = true; }
  });
  if (wall) {
    const T rho_w = sum / (T(1) + coef);
    static_for<1, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      constexpr int O = Lat<Q>::t.opp[I];
      const int t = matrix_target<Lat<Q>::t.cx[I], Lat<Q>::t.cy[I]>(a, p, x, y);
      if (t < 0) S[I] -= matrix_vbb<Q, T, O>(p, -1 - t, rho_w);
    });
  }
}

// Stores the canonical state S of the cell at (x, y) in layout a.parity.
template <int Q, typename T>
__device__ __forceinline__ void matrix_store_state(const MatrixArgs& a, const ModelParams& p, int x, int y, const T (&S)[Q]) {
  T* __restrict__ A = (T*)a.A;
  const long long ps = a.ps;
  const int c = y * a.nx + x;
  T rho_w = T(0);
#pragma unroll
  for (int i = 0; i < Q; ++i) rho_w += S[i];
  static_for<0, Q>([&](auto ic) {
    constexpr int I = decltype(ic)::value;
    constexpr int O = Lat<Q>::t.opp[I];
    const int t = matrix_target<Lat<Q>::t.cx[I], Lat<Q>::t.cy[I]>(a, p, x, y);
    if (t < 0) A[O * ps + c] = S[I] + matrix_vbb<Q, T, O>(p, -1 - t, rho_w);
    else if (a.parity == 0) A[I * ps + t] = S[I];
    else A[O * ps + c] = S[I];
  });
}

// lbm_init_fields: equilibrium of the given fields at the cell's own centre, stored in layout P0
template <int Q, typename T, int COLL>
__global__ void __launch_bounds__(128) matrix_init_kernel(const MatrixArgs a, const ModelParams p) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;      // storage index of the ABI
  if (c >= a.n) return;
  const int r = a.pos[c], y = r / a.nx, x = r - y * a.nx;
  T f[Q], g[Q], lam[NLAMBDA];
  equilibrium<Q, T, COLL, false>(p, T(a.rho[c]), T(a.ux[c]), T(a.uy[c]), T(cs2_v<Q>), lam, f, g);
  T s = T(0);
#pragma unroll
  for (int i = 0; i < Q; ++i) s += f[i];
  if (!(s > T(0)) || !isfinite(s)) atomicOr(a.status, FLAG_UNSTABLE);
  matrix_store_state<Q, T>(a, p, x, y, f);
}

// rho, u of the canonical state (Eq. 51 does not apply: athermal, T = c_s^2); output slot t = storage cell t or probe cells[t]
template <int Q, typename T, int COLL>
__global__ void __launch_bounds__(128) matrix_macro_kernel(const MatrixArgs a, const ModelParams p) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= a.n) return;
  const int c = a.cells ? a.cells[t] : t;
  const int r = a.pos[c], y = r / a.nx, x = r - y * a.nx;
  T S[Q], g[Q];
  matrix_load_state<Q, T>(a, p, x, y, S);
  T rho, ux, uy, Tm;
  moments<Q, T, false, false>(p, S, g, rho, ux, uy, Tm);
  a.o_rho[t] = (double)rho; a.o_ux[t] = (double)ux; a.o_uy[t] = (double)uy; a.o_T[t] = (double)Tm;
}

// eps of Eq. 52 of the canonical state (lbm_get_sensor); output slot = storage cell
template <int Q, typename T, int COLL>
__global__ void __launch_bounds__(128) matrix_sensor_kernel(const MatrixArgs a, const ModelParams p) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.n) return;
  const int r = a.pos[c], y = r / a.nx, x = r - y * a.nx;
  T S[Q], g[Q], lam[NLAMBDA];
  matrix_load_state<Q, T>(a, p, x, y, S);
  a.o_rho[c] = (double)sensor_of_state<Q, T, COLL, false>(p, S, g, lam);
}

// canonical-order population I/O of the parity tests: pops[storage cell][Q]
template <int Q, typename T, bool IMPORT>
__global__ void __launch_bounds__(128) matrix_io_kernel(const MatrixArgs a, const ModelParams p) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.n) return;
  const int r = a.pos[c], y = r / a.nx, x = r - y * a.nx;
  T S[Q];
  if constexpr (IMPORT) {
#pragma unroll
    for (int i = 0; i < Q; ++i) S[i] = (T)a.pops[(long long)c * Q + i];
    matrix_store_state<Q, T>(a, p, x, y, S);
  } else {
    matrix_load_state<Q, T>(a, p, x, y, S);
#pragma unroll
    for (int i = 0; i < Q; ++i) a.pops[(long long)c * Q + i] = (double)S[i];
  }
}

template <int Q, typename T, int COLL>
KernelSet with_matrix(KernelSet k, const char* name) {
  k.matrix_step[0][0] = (const void*)&matrix_step_kernel<Q, T, COLL, false, 1>;
  k.matrix_step[0][1] = (const void*)&matrix_step_kernel<Q, T, COLL, true, 1>;
  k.matrix_step[1][0] = (const void*)&matrix_step_kernel<Q, T, COLL, false, MATRIX_CPT<Q, T>>;
  k.matrix_step[1][1] = (const void*)&matrix_step_kernel<Q, T, COLL, true, MATRIX_CPT<Q, T>>;
  k.matrix_cpt = MATRIX_CPT<Q, T>;
  k.matrix_init = (const void*)&matrix_init_kernel<Q, T, COLL>;
  k.matrix_macro = (const void*)&matrix_macro_kernel<Q, T, COLL>;
  k.matrix_sensor = (const void*)&matrix_sensor_kernel<Q, T, COLL>;
  k.matrix_export = (const void*)&matrix_io_kernel<Q, T, false>;
  k.matrix_import = (const void*)&matrix_io_kernel<Q, T, true>;
  k.matrix_name = name;
  return k;
}

// an athermal polynomial kernel set with the matrix-like path beside the tree-stored one (lbm_config.addressing = LBM_ADDR_MATRIX)
#define LBM_KSET_MATRIX(Q, T, COLL) \
  with_matrix<Q, T, COLL>(LBM_KSET(Q, T, COLL, false, false), "matrix_step_kernel<" #Q "," #T "," #COLL "> (Cartesian index, AA pattern)")

}  // namespace lbm
