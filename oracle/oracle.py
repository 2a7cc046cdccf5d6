"""ctypes wrapper over the CPU ORACLE (oracle/*.c) -- test infrastructure, NOT the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares nothing with paper_2504_04465_b200 (the CUDA path).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = ["physics.c", "grid.c", "sim.c", "amr.c"]
_LIB = os.path.join(_HERE, "liboracle.so")

BGK, RR, NUMEQ = 0, 1, 2
BC_PERIODIC, BC_WALL, BC_MOVING_WALL, BC_INFLOW_VBB, BC_DIRICHLET_EQ, BC_DIRICHLET_EQ_RHO_EXTRAP, BC_NEUMANN = range(7)
FLUID, FINE_GHOST, COARSE_GHOST, NEUMANN, DIRICHLET = range(5)
LINK_NONE, LINK_WALL, LINK_VBB0 = -1, -2, -3


def build(force=False):
    """Compile liboracle.so with gcc (plain C11, -O2, no FMA contraction)."""
    srcs = [os.path.join(_HERE, s) for s in _SRC]
    deps = srcs + [os.path.join(_HERE, "oracle.h"), os.path.join(_HERE, "internal.h")]
    if not force and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(d) for d in deps):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-o", _LIB] + srcs + ["-lm"]
    subprocess.check_call(cmd)
    return _LIB


class OrcConfig(C.Structure):
    _fields_ = [
        ("lattice", C.c_int), ("collision", C.c_int), ("ddf", C.c_int), ("sensor", C.c_int),
        ("trace_eq", C.c_int), ("depth", C.c_int), ("nx_coarse", C.c_int), ("ny_coarse", C.c_int),
        ("newton_max_iter", C.c_int), ("bc", C.c_int * 4),
        ("tau0", C.c_double), ("T0", C.c_double), ("gamma", C.c_double), ("sensor_A", C.c_double),
        ("newton_tol", C.c_double),
        ("bc_rho", C.c_double * 4), ("bc_ux", C.c_double * 4), ("bc_uy", C.c_double * 4), ("bc_T", C.c_double * 4),
        ("sponge_x0", C.c_double), ("sponge_y0", C.c_double), ("sponge_r0", C.c_double), ("sponge_r1", C.c_double),
        ("sponge_sigma_max", C.c_double), ("sponge_rho_inf", C.c_double),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        vp, i64p, i32p, dp = C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32), C.POINTER(C.c_double)
        L.orc_grid_create.argtypes = [C.POINTER(OrcConfig), vp, vp, vp, vp, C.POINTER(vp)]
        L.orc_grid_destroy.argtypes = [vp]
        L.orc_grid_destroy.restype = None
        L.orc_num_cells.argtypes = [vp, C.c_int]
        L.orc_num_cells.restype = C.c_int64
        L.orc_num_ghosts.argtypes = [vp, C.c_int]
        L.orc_num_ghosts.restype = C.c_int64
        L.orc_tau.argtypes = [vp, C.c_int]
        L.orc_tau.restype = C.c_double
        L.orc_set_tau0.argtypes = [vp, C.c_double]
        L.orc_get_sponge.argtypes = [vp, C.c_int, vp]
        L.orc_set_bc_state.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double]
        L.orc_newton_iterations.argtypes = [vp]
        L.orc_newton_iterations.restype = C.c_int64
        L.orc_cell_updates.argtypes = [vp]
        L.orc_cell_updates.restype = C.c_int64
        L.orc_get_cells.argtypes = [vp, C.c_int, vp, vp, vp, vp]
        L.orc_get_nbr.argtypes = [vp, C.c_int, vp]
        L.orc_get_ghosts.argtypes = [vp, C.c_int, vp, vp, vp]
        L.orc_get_schedule.argtypes = [vp, vp, vp, C.c_int]
        L.orc_init_fields.argtypes = [vp, vp, vp, vp, vp]
        L.orc_step.argtypes = [vp, C.c_int]
        L.orc_step_fine.argtypes = [vp, C.c_int]
        L.orc_get_macroscopic.argtypes = [vp, vp, vp, vp, vp]
        L.orc_get_sensor.argtypes = [vp, vp]
        L.orc_get_populations.argtypes = [vp, C.c_int, C.c_int, vp]
        L.orc_set_populations.argtypes = [vp, C.c_int, C.c_int, vp]
        L.orc_transfer.argtypes = [vp, vp]
        L.orc_set_fine_step.argtypes = [vp, C.c_int64]
        L.orc_lattice.argtypes = [C.c_int, vp, vp, vp, vp, vp, vp]
        L.orc_feq_poly.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, vp]
        L.orc_feq_numerical.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, vp, vp]
        L.orc_collide_cell.argtypes = [C.POINTER(OrcConfig), C.c_double, vp, vp, vp, vp, vp]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def make_config(lattice=9, collision=BGK, ddf=0, sensor=0, trace_eq=0, depth=0, nx_coarse=1, ny_coarse=1,
                tau0=0.6, T0=0.0, gamma=1.4, sensor_A=1.5, newton_tol=1e-12, newton_max_iter=50,
                bc=(0, 0, 0, 0), bc_rho=(1, 1, 1, 1), bc_ux=(0, 0, 0, 0), bc_uy=(0, 0, 0, 0), bc_T=(0, 0, 0, 0),
                sponge=None):
    """sponge: None or (x0, y0, r0, r1, sigma_max, rho_inf) of Eq. 10-11."""
    c = OrcConfig()
    if sponge is not None:
        (c.sponge_x0, c.sponge_y0, c.sponge_r0, c.sponge_r1, c.sponge_sigma_max, c.sponge_rho_inf) = [float(v) for v in sponge]
    c.lattice, c.collision, c.ddf, c.sensor, c.trace_eq = lattice, collision, ddf, sensor, trace_eq
    c.depth, c.nx_coarse, c.ny_coarse, c.newton_max_iter = depth, nx_coarse, ny_coarse, newton_max_iter
    c.tau0, c.T0, c.gamma, c.sensor_A, c.newton_tol = tau0, T0, gamma, sensor_A, newton_tol
    for s in range(4):
        c.bc[s] = int(bc[s])
        c.bc_rho[s], c.bc_ux[s], c.bc_uy[s], c.bc_T[s] = float(bc_rho[s]), float(bc_ux[s]), float(bc_uy[s]), float(bc_T[s])
    return c


def lattice(Q):
    cx = np.zeros(Q, np.int32); cy = np.zeros(Q, np.int32); w = np.zeros(Q); opp = np.zeros(Q, np.int32)
    cs2 = C.c_double(); reach = C.c_int()
    rc = lib().orc_lattice(Q, _ptr(cx), _ptr(cy), _ptr(w), _ptr(opp), C.addressof(cs2), C.addressof(reach))
    assert rc == 0
    return cx, cy, w, opp, cs2.value, reach.value


def feq_poly(Q, rho, ux, uy, T=0.0, thermal=0):
    f = np.zeros(Q)
    assert lib().orc_feq_poly(Q, rho, ux, uy, T, thermal, _ptr(f)) == 0
    return f


def feq_numerical(Q, rho, ux, uy, T, lam=None, tol=1e-12, max_iter=50):
    lam = np.zeros(8) if lam is None else np.array(lam, dtype=np.float64)
    f = np.zeros(Q)
    it = lib().orc_feq_numerical(Q, rho, ux, uy, T, tol, max_iter, _ptr(lam), _ptr(f))
    return f, lam, it


def collide_cell(cfg, tau, f, g=None, lam=None):
    Q = cfg.lattice
    f = np.ascontiguousarray(f, dtype=np.float64)
    g = np.zeros(Q) if g is None else np.ascontiguousarray(g, dtype=np.float64)
    lam = np.zeros(8) if lam is None else np.array(lam, dtype=np.float64)
    fo = np.zeros(Q); go = np.zeros(Q)
    it = lib().orc_collide_cell(C.byref(cfg), tau, _ptr(f), _ptr(g), _ptr(lam), _ptr(fo), _ptr(go))
    return fo, go, lam, it


def _flatten(levels, depth):
    """list over levels 0..depth of (n,2) int32 arrays (or None) -> (offsets[depth+2], flat pairs)."""
    off = np.zeros(depth + 2, np.int64)
    parts = []
    for l in range(depth + 1):
        a = None if levels is None or l >= len(levels) else levels[l]
        n = 0 if a is None else len(a)
        off[l + 1] = off[l] + n
        if n:
            parts.append(np.ascontiguousarray(a, dtype=np.int32).reshape(-1, 2))
    flat = np.concatenate(parts) if parts else np.zeros((0, 2), np.int32)
    return off, np.ascontiguousarray(flat)


class OracleGrid:
    """One oracle simulation: mesh (split / solid cells per level) + model config."""

    def __init__(self, cfg, split=None, solid=None):
        self.cfg = cfg
        self.Q = cfg.lattice
        self.depth = cfg.depth
        so, sx = _flatten(split, cfg.depth)
        zo, zx = _flatten(solid, cfg.depth)
        h = C.c_void_p()
        rc = lib().orc_grid_create(C.byref(cfg), _ptr(so), _ptr(sx), _ptr(zo), _ptr(zx), C.byref(h))
        if rc != 0:
            raise RuntimeError("orc_grid_create failed: %d" % rc)
        self.h = h
        self.n = [int(lib().orc_num_cells(h, l)) for l in range(self.depth + 1)]
        self.off = np.concatenate([[0], np.cumsum(self.n)]).astype(np.int64)
        self.ntot = int(self.off[-1])

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_grid_destroy(self.h)
            self.h = None

    def tau(self, l):
        return lib().orc_tau(self.h, l)

    def sponge(self, l):
        a = np.zeros(self.n[l])
        assert lib().orc_get_sponge(self.h, l, _ptr(a)) == 0
        return a

    def set_tau0(self, tau0):
        return lib().orc_set_tau0(self.h, float(tau0))

    def set_bc_state(self, side, rho, ux, uy, T=0.0):
        return lib().orc_set_bc_state(self.h, int(side), float(rho), float(ux), float(uy), float(T))

    def cells(self, l):
        n = self.n[l]
        ix = np.zeros(n, np.int32); iy = np.zeros(n, np.int32); ty = np.zeros(n, np.int32); aux = np.zeros(n, np.int32)
        assert lib().orc_get_cells(self.h, l, _ptr(ix), _ptr(iy), _ptr(ty), _ptr(aux)) == 0
        return ix, iy, ty, aux

    def nbr(self, l):
        a = np.zeros((self.n[l], self.Q - 1), np.int32)
        assert lib().orc_get_nbr(self.h, l, _ptr(a)) == 0
        return a

    def ghosts(self, l):
        ng = int(lib().orc_num_ghosts(self.h, l))
        co = np.zeros(ng, np.int32); ch = np.zeros((ng, 4), np.int32); m = np.zeros(ng, np.uint64)
        if ng:
            assert lib().orc_get_ghosts(self.h, l, _ptr(co), _ptr(ch), _ptr(m)) == 0
        return co, ch, m

    def schedule(self):
        n = lib().orc_get_schedule(self.h, None, None, 0)
        k = np.zeros(n, np.int32); lv = np.zeros(n, np.int32)
        lib().orc_get_schedule(self.h, _ptr(k), _ptr(lv), n)
        return k, lv

    def init_fields(self, rho, ux, uy, T=None):
        a = [np.ascontiguousarray(x, dtype=np.float64) for x in (rho, ux, uy)]
        t = None if T is None else np.ascontiguousarray(T, dtype=np.float64)
        for x in a:
            assert x.size == self.ntot
        return lib().orc_init_fields(self.h, _ptr(a[0]), _ptr(a[1]), _ptr(a[2]), _ptr(t))

    def step(self, n=1):
        return lib().orc_step(self.h, n)

    def step_fine(self, n=1):
        return lib().orc_step_fine(self.h, n)

    def macroscopic(self):
        r = np.zeros(self.ntot); u = np.zeros(self.ntot); v = np.zeros(self.ntot); T = np.zeros(self.ntot)
        assert lib().orc_get_macroscopic(self.h, _ptr(r), _ptr(u), _ptr(v), _ptr(T)) == 0
        return r, u, v, T

    def sensor(self):
        """eps of Eq. 52 of the current state of every stored cell, flat over the levels (orc_get_sensor)."""
        e = np.zeros(self.ntot)
        rc = lib().orc_get_sensor(self.h, _ptr(e))
        if rc != 0:
            raise RuntimeError("orc_get_sensor: %d" % rc)
        return e

    def populations(self, l, which=0):
        cnt = 8 if which == 2 else self.Q
        a = np.zeros((self.n[l], cnt))
        rc = lib().orc_get_populations(self.h, l, which, _ptr(a))
        if rc != 0:
            raise RuntimeError("orc_get_populations: %d" % rc)
        return a

    def set_populations(self, l, which, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        rc = lib().orc_set_populations(self.h, l, which, _ptr(a))
        if rc != 0:
            raise RuntimeError("orc_set_populations: %d" % rc)

    def set_fine_step(self, k):
        return lib().orc_set_fine_step(self.h, int(k))

    def transfer_from(self, src):
        """orc_transfer: takes over the state of `src` (another tree over the same box), Sec. 8.1 of the paper."""
        return lib().orc_transfer(self.h, src.h)

    def newton_iterations(self):
        return int(lib().orc_newton_iterations(self.h))

    def cell_updates(self):
        return int(lib().orc_cell_updates(self.h))
