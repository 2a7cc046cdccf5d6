// sweep_pipe.cuh -- software-pipelined level sweep for the wide models (second distribution g and / or numerical
// equilibria: rows a1-a9 of SURVEY.md Sec. 8(a), the same cell update as sweep.cuh's list path).
//
// Why a second kernel.  The wide models hold 42-82 reals per cell and their arithmetic needs 160-255 registers, so only
// 8 warps are resident per SM; ncu (profiles/r02_ncu_naca_f64.md, r02_ncu_riemann_f64.md, r02_ncu_sod21_f32.md) shows those
// warps waiting on their own gathers (stall_long_scoreboard 1.6-2.8 cycles per issued instruction, fp64 pipe 29-37 % busy,
// DRAM 43-60 %): one cell per thread means gather -> wait -> compute -> store, and two warps per scheduler cannot hide a
// DRAM round trip behind each other's arithmetic.  Here a CTA walks over many tiles of TPB consecutive cells (persistent
// grid: every resident CTA slot of the device once; tiles handed out in Z-curve order from a per-level counter) and a
// thread keeps the NEXT cell's gathers in flight while it computes the current one:
//   pass p:  request the id of the tile after next (atomicAdd, consumed at the end of the pass);
//            cp.async.wait_group 0: the stage of cell p and the links of cell p+1 have landed;
//            issue the gathers of cell p+1 as cp.async (LDGSTS) into shared-memory stage (p+1)&1 from those links, then
//            the links of cell p+2 into the link slots;  compute cell p out of stage p&1;  store;
//            publish the new tile id, one __syncthreads().
// A thread reads and writes only its own shared-memory slots (plane-major, [stage][plane][thread]: conflict-free 4 / 8-byte
// accesses), and the populations of the current cell stay in shared memory (streamed through the moment, sensor and
// relaxation passes) instead of in registers; no register holds a link or a population across the arithmetic.  Cell
// types are handled as in sweep.cuh; the rare ones (coarse ghosts: coalescence, explosion; Dirichlet cells) patch their
// stage in place with synchronous loads.  Velocity bounce-back links do not occur (weakly compressible models only,
// lbm_grid_create rejects them here).  The last CTA to finish zeroes the counters, so every launch finds an empty queue; the
// kernel is launched without a programmatic edge (the queue must not be touched while the previous launch on the level runs).
#pragma once
#include "sweep.cuh"

namespace lbm {

template <int Q, typename T, int COLL, bool DDF>
struct PipeCfg {
  using PL = PopLayout<Q, DDF, COLL>;
  static constexpr int STAGES = 2;
  // per thread: two stages of NPOP reals + one row of Q-1 links (int32) of the cell after
  static constexpr int bytes_per_thread = STAGES * PL::NPOP * (int)sizeof(T) + (Q - 1) * 4;
  // 128 threads per CTA where two CTAs fit the 228 KB of an SM (1 KB per CTA is the system's), else 64 (D2Q37 in fp64)
  static constexpr int SM_BYTES = 228 * 1024;
  static constexpr int TPB = (2 * (128 * bytes_per_thread + 1024) <= SM_BYTES) ? 128 : 64;
  static constexpr int smem = TPB * bytes_per_thread;
  static constexpr int by_smem = SM_BYTES / (smem + 1024);
  // resident CTAs per SM asked of ptxas (register cap = 65536 / (TPB * CTAS)): two for the fp64 Newton solve (255
  // registers), up to four x 128 threads otherwise
  static constexpr int want = (COLL == LBM_NUMEQ && sizeof(T) == 8) ? 2 : (512 / TPB);
  static constexpr int CTAS = by_smem < want ? by_smem : want;
};

__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
template <typename T>
__device__ __forceinline__ void cp_async_one(unsigned dst, const T* src) {
  static_assert(sizeof(T) == 4 || sizeof(T) == 8, "cp.async element size");
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst), "l"(src), "n"((int)sizeof(T)) : "memory");
}

template <int Q, typename T, int COLL, bool DDF, bool SENSOR>
__global__ void __launch_bounds__((PipeCfg<Q, T, COLL, DDF>::TPB), (PipeCfg<Q, T, COLL, DDF>::CTAS))
sweep_pipe_kernel(const LevelArgs a, const ModelParams p) {
  using PL = PopLayout<Q, DDF, COLL>;
  using PC = PipeCfg<Q, T, COLL, DDF>;
  constexpr bool NUMEQ = COLL == LBM_NUMEQ;
  constexpr int TPB = PC::TPB, NPOP = PL::NPOP;
  static_assert(DDF || NUMEQ, "the pipelined sweep is instantiated for the wide models only");
  static_assert(COLL != LBM_RR, "RR is athermal");
  extern __shared__ __align__(16) unsigned char pipe_smem[];
  // shared memory, all of it private to its thread: plane q of stage s at sm[(s * NPOP + q) * TPB], then link I (1..Q-1)
  // of the cell whose gathers are issued next at lks[(I - 1) * TPB]
  T* const sm = reinterpret_cast<T*>(pipe_smem) + threadIdx.x;
  const int* const lks = reinterpret_cast<const int*>(pipe_smem + PC::STAGES * NPOP * TPB * sizeof(T)) + threadIdx.x;
  const unsigned sm_addr = (unsigned)__cvta_generic_to_shared(sm);
  const unsigned lk_addr = (unsigned)__cvta_generic_to_shared(lks);
  pdl_launch_dependents();
  const T* __restrict__ So = (const T*)a.So;
  T* __restrict__ Sn = (T*)a.Sn;
  long long ps = a.ps;      // laundered once per pass (below), so that no address is hoisted out of the cell loop
  const int n = a.n;

  // a cell's descriptor: storage index, cell whose own values it reads (itself; a Neumann cell: its source, S13),
  // type byte, aux, mask of NONE links
  struct Desc { int c, self, tb, aux; unsigned long long none; };

  // links of cell c -> the thread's link slots (cp.async: no register holds them across the compute phase; the links
  // are static tables, so this may run before the previous sweep has drained, PDL)
  auto issue_links = [&](int c) {
    static_for<1, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      cp_async_one(lk_addr + (unsigned)((I - 1) * TPB * 4), a.nbr + (long long)(I - 1) * ps + c);
    });
  };
  // issues the gathers of cell c (its links are in the link slots, its type byte in tb) into stage s; returns its descriptor
  auto issue = [&](int c, int tb, int s) -> Desc {
    Desc d;
    d.c = c; d.tb = tb; d.aux = -1; d.none = 0ull;
    const int type = tb & TYPE_MASK;
    if (type != LBM_FLUID && type != LBM_FINE_GHOST) d.aux = a.aux[c];
    d.self = (type == LBM_NEUMANN) ? d.aux : c;
    const unsigned st = sm_addr + (unsigned)(s * NPOP * TPB * (int)sizeof(T));
    cp_async_one(st, So + d.self);
    if constexpr (DDF) cp_async_one(st + (unsigned)(PL::G0 * TPB * (int)sizeof(T)), So + PL::G0 * ps + d.self);
    static_for<1, Q>([&](auto ic) {
      constexpr int I = decltype(ic)::value;
      constexpr int O = Lat<Q>::t.opp[I];
      const int l = lks[(I - 1) * TPB];
      // pull form of Eq. 31, branch-free: a wall link reads the cell's own opposite population, a NONE link
      // the cell's own value (fine ghosts, S6; coarse ghosts: coalesced below), any other link the neighbour's
      const int src = l >= 0 ? l : d.self;
      const bool same = l >= 0 || l == LBM_LINK_NONE;
      if (l == LBM_LINK_NONE) d.none |= 1ull << I;
      cp_async_one(st + (unsigned)(I * TPB * (int)sizeof(T)), (same ? So + I * ps : So + O * ps) + src);
      if constexpr (DDF)
        cp_async_one(st + (unsigned)((PL::G0 + I) * TPB * (int)sizeof(T)), (same ? So + (PL::G0 + I) * ps : So + (PL::G0 + O) * ps) + src);
    });
    if constexpr (NUMEQ) {
#pragma unroll
      for (int k = 0; k < NLAMBDA; ++k)
        cp_async_one(st + (unsigned)((PL::L0 + k) * TPB * (int)sizeof(T)), So + (PL::L0 + k) * ps + d.self);
    }
    return d;
  };

  [[maybe_unused]] unsigned n_steps = 0u, n_solves = 0u;
  // ---- tile queue.  Tiles of TPB consecutive cells are handed out in Z-curve order from one counter per level, the order
  // in which the hardware would start the CTAs of a one-cell-per-thread launch: tiles that are neighbours in space are
  // gathered at about the same time whatever their cells cost (Newton counts differ), so warps that share DRAM sectors
  // still meet in the L2.  (With a fixed stride per thread the CTAs drifted apart: +47 % DRAM reads.)  The id a CTA needs
  // two passes later is requested at the top of a pass and published at its end; one block barrier per pass, which also
  // keeps the four warps of a CTA in the same stretch of code.
  __shared__ int s_tile[2];
  int* const q_ctr = a.queue;
  int* const q_done = a.queue + 1;
  const int n_tiles = (n + TPB - 1) / TPB;
  if (threadIdx.x == 0) { s_tile[0] = atomicAdd(q_ctr, 1); s_tile[1] = atomicAdd(q_ctr, 1); }
  __syncthreads();
  int t_n = s_tile[0], t_nn = s_tile[1];                   // tile whose gathers are issued next, tile after it (CTA-uniform)
  __syncthreads();
  int cn = t_n < n_tiles ? t_n * TPB + (int)threadIdx.x : n;   // the cell whose gathers are issued next
  int tb_n = 0;                                            // its type byte (one register carried across the compute phase)
  Desc cur;
  cur.c = n;                                               // nothing to compute in the first pass
  if (cn < n) { issue_links(cn); tb_n = a.type[cn]; }
  cp_async_commit();
  pdl_wait();      // from here on: data written by the previous sweeps of the stream
  int s = 0, pass = 0;
#pragma unroll 1
  for (;;) {
    int req = 0;
    if (threadIdx.x == 0) req = atomicAdd(q_ctr, 1);       // in flight during this pass
    // ---- keep the pipeline full.  Everything issued so far has landed after this wait: stage s (the cell to compute
    // now, issued one pass ago and in flight during the previous cell's arithmetic) and the link slots.  Then: gathers of
    // the next cell into the other stage, links of the cell after into the link slots (after the gathers that read them).
    cp_async_wait<0>();
    // the 2 NPOP plane addresses (base + plane * ps) are loop invariants the compiler would otherwise keep in ~200 registers
    // and spill (the stack sits in an L1 that this kernel's shared memory leaves ~20 KB of); one multiply-add each instead
    asm volatile("" : "+l"(ps));
    Desc nxt;
    nxt.c = n;
    if (cn < n) nxt = issue(cn, tb_n, s ^ 1);
    const int cnn = t_nn < n_tiles ? t_nn * TPB + (int)threadIdx.x : n;
    if (cnn < n) { issue_links(cnn); tb_n = a.type[cnn]; }
    cp_async_commit();

    if (cur.c < n) {
    // ---- the cell update out of stage s
    T* const st = sm + s * NPOP * TPB;
    const int c = cur.c;
    const int type = cur.tb & TYPE_MASK;
    Imposed<T> imp{false, T(0), T(0), T(0), T(0)};
    bool collide_it = true;
    if (type == LBM_FINE_GHOST) {
      // fine ghost cells stream without colliding; lambda stays
#pragma unroll
      for (int q = 0; q < NPOP; ++q) Sn[q * ps + c] = st[q * TPB];
      collide_it = false;
    } else if (type == LBM_DIRICHLET) {
      // equilibrium Dirichlet cell: imposed (rho,u,T); rho optionally from the nearest interior cell
      const int sd = cur.tb >> TYPE_SIDE_SHIFT;
      T rho = T(p.bc_rho[sd]);
      if (p.bc_kind[sd] == LBM_BC_DIRICHLET_EQ_RHO_EXTRAP) {
        rho = T(0);
#pragma unroll
        for (int i = 0; i < Q; ++i) rho += So[i * ps + cur.aux];
      }
      imp = Imposed<T>{true, rho, T(p.bc_ux[sd]), T(p.bc_uy[sd]), T(p.bc_T[sd])};
      if (!(rho > T(0)) || !isfinite(rho)) atomicOr(a.status, FLAG_UNSTABLE);
    } else if (type == LBM_COARSE_GHOST) {
      const int* ch = a.g_child + 4ll * cur.aux;
      const int k0 = ch[0], k1 = ch[1], k2 = ch[2], k3 = ch[3];
      const T nf = T((k0 >= 0) + (k1 >= 0) + (k2 >= 0) + (k3 >= 0));
      const T* F = (const T*)a.fine;
      const long long fps = a.fps;
      if (cur.none != 0ull) {
        // coalescence (Eq. 4): unknown directions only, mean over the children that exist
        static_for<1, Q>([&](auto ic) {
          constexpr int I = decltype(ic)::value;
          if ((cur.none >> I) & 1ull) {
            T sf = T(0);
            if (k0 >= 0) sf += F[I * fps + k0];
            if (k1 >= 0) sf += F[I * fps + k1];
            if (k2 >= 0) sf += F[I * fps + k2];
            if (k3 >= 0) sf += F[I * fps + k3];
            st[I * TPB] = sf / nf;
            if constexpr (DDF) {
              T sg = T(0);
              if (k0 >= 0) sg += F[(PL::G0 + I) * fps + k0];
              if (k1 >= 0) sg += F[(PL::G0 + I) * fps + k1];
              if (k2 >= 0) sg += F[(PL::G0 + I) * fps + k2];
              if (k3 >= 0) sg += F[(PL::G0 + I) * fps + k3];
              st[(PL::G0 + I) * TPB] = sg / nf;
            }
          }
        });
      }
      if constexpr (NUMEQ) {      // Eq. 6: warm start from the mean of the children's multipliers
#pragma unroll
        for (int k = 0; k < NLAMBDA; ++k) {
          T sl = T(0);
          if (k0 >= 0) sl += F[(PL::L0 + k) * fps + k0];
          if (k1 >= 0) sl += F[(PL::L0 + k) * fps + k1];
          if (k2 >= 0) sl += F[(PL::L0 + k) * fps + k2];
          if (k3 >= 0) sl += F[(PL::L0 + k) * fps + k3];
          st[(PL::L0 + k) * TPB] = sl / nf;
        }
      }
    }

    if (collide_it) {
      // ---- steps 2-5 streamed out of the stage: moments, equilibrium, sensor, relaxation + store
      T rho = T(0), jx = T(0), jy = T(0), e2 = T(0);
      static_for<0, Q>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        constexpr int cx = Lat<Q>::t.cx[I], cy = Lat<Q>::t.cy[I], xi2 = cx * cx + cy * cy;
        const T fi = st[I * TPB];
        rho += fi;
        if constexpr (cx != 0) jx += T(cx) * fi;
        if constexpr (cy != 0) jy += T(cy) * fi;
        if constexpr (DDF) e2 += T(xi2) * fi + st[(PL::G0 + I) * TPB];
        else if constexpr (xi2 != 0) e2 += T(xi2) * fi;
      });
      T ux = jx / rho, uy = jy / rho;
      const T Cv = DDF ? T(1.0 / (p.gamma - 1.0)) : T(1);
      T Tm = (e2 - rho * (ux * ux + uy * uy)) / (T(2) * rho * Cv);                  // Eq. 51
      if (imp.on) { rho = imp.rho; ux = imp.ux; uy = imp.uy; Tm = imp.Tm; }
      if (!(rho > T(0)) || !isfinite(rho)) atomicOr(a.status, FLAG_UNSTABLE);
      const T fac = DDF ? T(2.0 / (p.gamma - 1.0) - 2.0) * Tm : T(0);                 // Eq. 50: (2 C_v - D) T
      const T tau = T(a.tau);
      if constexpr (NUMEQ) {
        T lam[NLAMBDA], feq[Q];
#pragma unroll
        for (int k = 0; k < NLAMBDA; ++k) lam[k] = st[(PL::L0 + k) * TPB];
        const int it = feq_numerical<Q, T>(p, rho, ux, uy, Tm, lam, feq);
        n_steps += newton_steps(it); n_solves += 1u;
        if (it < 0) atomicOr(a.status, FLAG_NEWTON);
        T tau_eff = tau;
        if constexpr (SENSOR) {
          T eps = T(0);
#pragma unroll
          for (int i = 0; i < Q; ++i) {
            T den = Num<T>::abs_(feq[i]);
            if (den < Num<T>::tiny()) den = Num<T>::tiny();
            eps += Num<T>::abs_(st[i * TPB] - feq[i]) * fast_rcp(den);            // Eq. 52
          }
          eps /= T(Q);
          tau_eff = tau * sensor_alpha<T>(eps, T(p.sensor_A), tau);
        }
        const T keep = T(1) - T(1) / tau_eff;
#pragma unroll
        for (int i = 0; i < Q; ++i) {
          Sn[i * ps + c] = imp.on ? feq[i] : feq[i] + keep * (st[i * TPB] - feq[i]);                  // Eq. 30
          if constexpr (DDF) { const T ge = fac * feq[i]; Sn[(PL::G0 + i) * ps + c] = imp.on ? ge : ge + keep * (st[(PL::G0 + i) * TPB] - ge); }
        }
#pragma unroll
        for (int k = 0; k < NLAMBDA; ++k) Sn[(PL::L0 + k) * ps + c] = lam[k];
      } else {
        T am[NA];
        aeq_moments<T>(rho, ux, uy, Tm - T(cs2_v<Q>), am);
        T keep = T(1) - T(1) / tau;
        if constexpr (SENSOR) {
          T eps = T(0);
          poly_all<Q, T>(am, [&](auto ic, T fe) {
            constexpr int I = decltype(ic)::value;
            T den = Num<T>::abs_(fe);
            if (den < Num<T>::tiny()) den = Num<T>::tiny();
            eps += Num<T>::abs_(st[I * TPB] - fe) * fast_rcp(den);                // Eq. 52
          });
          eps /= T(Q);
          keep = T(1) - T(1) / (tau * sensor_alpha<T>(eps, T(p.sensor_A), tau));
#pragma unroll
          for (int k = 0; k < NA; ++k) opaque(am[k]);     // f^eq is recomputed, not kept (see collide.cuh)
        }
        poly_all<Q, T>(am, [&](auto ic, T fe) {
          constexpr int I = decltype(ic)::value;
          Sn[I * ps + c] = imp.on ? fe : fe + keep * (st[I * TPB] - fe);
          const T ge = fac * fe;
          Sn[(PL::G0 + I) * ps + c] = imp.on ? ge : ge + keep * (st[(PL::G0 + I) * TPB] - ge);
        });
      }

      if (type == LBM_COARSE_GHOST) {
        // uniform explosion (Eq. 5, 7): every child receives the coarse post-collision state, all directions (S8);
        // the state is read back from this thread's own stores
        const int* ch = a.g_child + 4ll * cur.aux;
        T* F = (T*)a.fine;
        const long long fps = a.fps;
#pragma unroll 1
        for (int q = 0; q < NPOP; ++q) {
          const T v = Sn[q * ps + c];
          for (int k = 0; k < 4; ++k) {
            const int cq = ch[k];
            if (cq >= 0) F[q * fps + cq] = v;
          }
        }
      }
    }
    }     // cur.c < n
    if (t_n >= n_tiles) break;       // CTA-uniform: nothing was issued in this pass, the queue is empty
    if (threadIdx.x == 0) s_tile[pass & 1] = req;
    __syncthreads();
    const int t_new = s_tile[pass & 1];
    cur = nxt; cn = cnn; t_n = t_nn; t_nn = t_new; s ^= 1; ++pass;
  }
  cp_async_wait<0>();
  // the last CTA out leaves the queue ready for the next launch on this level
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    if (atomicAdd(q_done, 1) == (int)gridDim.x - 1) { atomicExch(q_ctr, 0); atomicExch(q_done, 0); }
  }
  if constexpr (NUMEQ) {
    __syncwarp();
    count_newton(a.status, n_steps, n_solves);
  }
}

template <int Q, typename T, int COLL, bool DDF, bool SENSOR>
KernelSet make_kernel_set_pipe(const char* name, const char* bricks_name, const char* pipe_name) {
  using PC = PipeCfg<Q, T, COLL, DDF>;
  KernelSet k = make_kernel_set<Q, T, COLL, DDF, SENSOR>(name, bricks_name);
  k.sweep_pipe = (const void*)&sweep_pipe_kernel<Q, T, COLL, DDF, SENSOR>;
  k.pipe_name = pipe_name;
  k.pipe_tpb = PC::TPB;
  k.pipe_smem = PC::smem;
  // Measured on one B200 (GLUPS, pipelined / one cell per thread): Sod D2Q13 fp32 11.3 / 10.0, Sod D2Q21
  // fp32 7.9 / 7.7, Sod D2Q37 fp32 3.0 / 3.5, Sod D2Q21 fp64 3.5 / 4.9, naca fp64 2.9 / 4.3: the gather stalls are gone
  // (stall_long_scoreboard 1.6 -> 0.2 per issue, Sod D2Q21 fp32), but the fp32 solves are instruction-bound either way
  // and the fp64 ones pay for the 20 KB of L1 this kernel's shared memory leaves them; AUTO selects it where it wins clearly.
  k.pipe_auto = (COLL == LBM_NUMEQ && sizeof(T) == 4 && Q == 13) ? 1 : 0;
  return k;
}

// a kernel set whose large levels run the pipelined sweep (the one-cell-per-thread kernels stay for small levels and as
// the A/B reference, lbm_config.no_pipeline)
#define LBM_KSET_PIPE(Q, T, COLL, DDF, SENSOR) \
  make_kernel_set_pipe<Q, T, COLL, DDF, SENSOR>("sweep_kernel<" #Q "," #T "," #COLL "," #DDF "," #SENSOR ",false>", \
                                                "sweep_kernel<" #Q "," #T "," #COLL "," #DDF "," #SENSOR ",true> (bricks + list)", \
                                                "sweep_pipe_kernel<" #Q "," #T "," #COLL "," #DDF "," #SENSOR "> (pipelined)")

}  // namespace lbm
