"""Thin ctypes binding over the C ABI of include/lbm.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of liblbm_b200.so; PyTorch is used for the device
arena and the stream only.  There is no CPU fallback: importing this module raises if the library has
not been built (`python -m paper_2504_04465_b200.build`), and binding a grid raises without a CUDA device.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblbm_b200.so")

MAX_LEVELS = 24
BGK, RR, NUMEQ = 0, 1, 2
ADDR_AUTO, ADDR_LIST, ADDR_BRICKS, ADDR_MATRIX = 0, 1, 2, 3
PIPE_AUTO, PIPE_OFF, PIPE_ALWAYS = 0, 1, 2
BC_PERIODIC, BC_WALL, BC_MOVING_WALL, BC_INFLOW_VBB, BC_DIRICHLET_EQ, BC_DIRICHLET_EQ_RHO_EXTRAP, BC_NEUMANN = range(7)
FLUID, FINE_GHOST, COARSE_GHOST, NEUMANN, DIRICHLET = range(5)
LINK_NONE, LINK_WALL, LINK_VBB0 = -1, -2, -3
OK, EINVAL, ENOMEM, EMESH, ECUDA, EUNSTABLE, ENEWTON, EUNSUPPORTED, ESTATE, ETOOLARGE = 0, -1, -2, -3, -4, -5, -6, -7, -8, -9
STATIC_PROBE_MAX = 4096
_ERR = {EINVAL: "LBM_EINVAL", ENOMEM: "LBM_ENOMEM", EMESH: "LBM_EMESH", ECUDA: "LBM_ECUDA", EUNSTABLE: "LBM_EUNSTABLE",
        ENEWTON: "LBM_ENEWTON", EUNSUPPORTED: "LBM_EUNSUPPORTED", ESTATE: "LBM_ESTATE", ETOOLARGE: "LBM_ETOOLARGE"}

# every symbol include/lbm.h declares (checked by tests/test_abi.py)
SYMBOLS = ["lbm_grid_create", "lbm_destroy", "lbm_grid_query", "lbm_supported_model", "lbm_get_cells", "lbm_get_nbr", "lbm_get_ghosts",
           "lbm_get_schedule", "lbm_get_sponge", "lbm_get_bricks", "lbm_grid_bind", "lbm_init_fields", "lbm_step", "lbm_step_fine", "lbm_transfer", "lbm_set_relaxation", "lbm_set_boundary_state", "lbm_sync", "lbm_get_macroscopic", "lbm_get_macroscopic_at", "lbm_get_macroscopic_at_static", "lbm_get_sensor",
           "lbm_get_populations", "lbm_set_populations", "lbm_last_step_ms", "lbm_kernel_name", "lbm_newton_iterations", "lbm_measure_fma_peak"]


class LbmError(RuntimeError):
    def __init__(self, where, code):
        super().__init__("%s failed: %s (%d)" % (where, _ERR.get(code, "?"), code))
        self.code = code


class LbmConfig(C.Structure):
    _fields_ = [
        ("lattice", C.c_int), ("precision", C.c_int), ("collision", C.c_int), ("ddf", C.c_int), ("sensor", C.c_int),
        ("trace_eq", C.c_int), ("depth", C.c_int), ("nx_coarse", C.c_int), ("ny_coarse", C.c_int),
        ("newton_max_iter", C.c_int), ("bc", C.c_int * 4),
        ("tau0", C.c_double), ("T0", C.c_double), ("gamma", C.c_double), ("sensor_A", C.c_double),
        ("newton_tol", C.c_double),
        ("bc_rho", C.c_double * 4), ("bc_ux", C.c_double * 4), ("bc_uy", C.c_double * 4), ("bc_T", C.c_double * 4),
        ("sponge_x0", C.c_double), ("sponge_y0", C.c_double), ("sponge_r0", C.c_double), ("sponge_r1", C.c_double),
        ("sponge_sigma_max", C.c_double), ("sponge_rho_inf", C.c_double),
        ("addressing", C.c_int), ("no_pdl", C.c_int), ("pipeline", C.c_int), ("pipe_max_ctas", C.c_int), ("no_prefetch", C.c_int), ("concurrent_levels", C.c_int),
    ]


class LbmGridInfo(C.Structure):
    _fields_ = [
        ("depth", C.c_int), ("Q", C.c_int), ("W", C.c_int), ("npop", C.c_int), ("precision", C.c_int),
        ("n_cells", C.c_int64 * MAX_LEVELS), ("n_inbox", C.c_int64 * MAX_LEVELS),
        ("n_coarse_ghosts", C.c_int64 * MAX_LEVELS), ("n_fine_ghosts", C.c_int64 * MAX_LEVELS),
        ("n_total", C.c_int64), ("updates_per_coarse_step", C.c_int64), ("launches_per_coarse_step", C.c_int64),
        ("arena_bytes", C.c_size_t), ("tau", C.c_double * MAX_LEVELS), ("n_bricks", C.c_int64 * MAX_LEVELS),
        ("brick_min_level_cells", C.c_int64),
    ]


_lib = None


def lib():
    """Loads liblbm_b200.so; raises (no fallback) if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not built: run `python -m paper_2504_04465_b200.build` (there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.lbm_grid_create.argtypes = [C.POINTER(LbmConfig), vp, vp, vp, vp, C.POINTER(vp)]
        L.lbm_destroy.argtypes = [vp]
        L.lbm_destroy.restype = None
        L.lbm_grid_query.argtypes = [vp, C.POINTER(LbmGridInfo)]
        L.lbm_supported_model.argtypes = [C.c_int, C.POINTER(LbmConfig)]
        L.lbm_get_cells.argtypes = [vp, C.c_int, vp, vp, vp, vp]
        L.lbm_get_nbr.argtypes = [vp, C.c_int, vp]
        L.lbm_get_ghosts.argtypes = [vp, C.c_int, vp, vp, vp]
        L.lbm_get_schedule.argtypes = [vp, vp, vp, C.c_int]
        L.lbm_get_bricks.argtypes = [vp, C.c_int, vp, vp]
        L.lbm_get_sponge.argtypes = [vp, C.c_int, vp]
        L.lbm_grid_bind.argtypes = [vp, vp, C.c_size_t, vp]
        L.lbm_init_fields.argtypes = [vp, vp, vp, vp, vp]
        L.lbm_step.argtypes = [vp, C.c_int]
        L.lbm_step_fine.argtypes = [vp, C.c_int]
        L.lbm_set_relaxation.argtypes = [vp, C.c_double]
        L.lbm_set_boundary_state.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double]
        L.lbm_transfer.argtypes = [vp, vp]
        L.lbm_sync.argtypes = [vp]
        L.lbm_get_macroscopic.argtypes = [vp, vp, vp, vp, vp]
        L.lbm_get_macroscopic_at.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp, vp, vp]
        L.lbm_get_macroscopic_at_static.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp, vp, vp]
        L.lbm_get_sensor.argtypes = [vp, vp]
        L.lbm_get_populations.argtypes = [vp, C.c_int, C.c_int, vp]
        L.lbm_set_populations.argtypes = [vp, C.c_int, C.c_int, vp]
        L.lbm_last_step_ms.argtypes = [vp]
        L.lbm_last_step_ms.restype = C.c_double
        L.lbm_kernel_name.argtypes = [vp]
        L.lbm_kernel_name.restype = C.c_char_p
        L.lbm_newton_iterations.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.lbm_measure_fma_peak.argtypes = [C.c_int, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        _lib = L
    return _lib


def measure_fma_peak(precision=64, seconds=1.0):
    """lbm_measure_fma_peak: (TFLOP/s, FMA lanes x MHz per SM) of the current device's plain fp64 / fp32 pipe."""
    tf, lm = C.c_double(0.0), C.c_double(0.0)
    _check("lbm_measure_fma_peak", lib().lbm_measure_fma_peak(int(precision), float(seconds), C.byref(tf), C.byref(lm)))
    return tf.value, lm.value


def supported_models():
    """(lattice, precision, collision, ddf, sensor) of every compiled kernel set (lbm_supported_model)."""
    out, c, i = [], LbmConfig(), 0
    while lib().lbm_supported_model(i, C.byref(c)) == 0:
        out.append((c.lattice, c.precision, c.collision, c.ddf, c.sensor))
        i += 1
    return out


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(where, rc):
    if rc != 0:
        raise LbmError(where, rc)


def make_config(lattice=9, precision=64, collision=BGK, ddf=0, sensor=0, trace_eq=0, depth=0, nx_coarse=1, ny_coarse=1,
                tau0=0.6, T0=0.0, gamma=1.4, sensor_A=1.5, newton_tol=1e-12, newton_max_iter=50,
                bc=(0, 0, 0, 0), bc_rho=(1, 1, 1, 1), bc_ux=(0, 0, 0, 0), bc_uy=(0, 0, 0, 0), bc_T=(0, 0, 0, 0),
                sponge=None, addressing=ADDR_AUTO, no_pdl=0, pipeline=0, pipe_max_ctas=0, no_prefetch=0, concurrent_levels=0):
    """sponge: None or (x0, y0, r0, r1, sigma_max, rho_inf) of Eq. 10-11; addressing, no_pdl, pipeline, pipe_max_ctas: device-path options."""
    c = LbmConfig()
    c.addressing, c.no_pdl, c.pipeline, c.pipe_max_ctas, c.no_prefetch = int(addressing), int(no_pdl), int(pipeline), int(pipe_max_ctas), int(no_prefetch)
    c.concurrent_levels = int(concurrent_levels)
    if sponge is not None:
        (c.sponge_x0, c.sponge_y0, c.sponge_r0, c.sponge_r1, c.sponge_sigma_max, c.sponge_rho_inf) = [float(v) for v in sponge]
    c.lattice, c.precision, c.collision, c.ddf, c.sensor, c.trace_eq = lattice, precision, collision, ddf, sensor, trace_eq
    c.depth, c.nx_coarse, c.ny_coarse, c.newton_max_iter = depth, nx_coarse, ny_coarse, newton_max_iter
    c.tau0, c.T0, c.gamma, c.sensor_A, c.newton_tol = tau0, T0, gamma, sensor_A, newton_tol
    for s in range(4):
        c.bc[s] = int(bc[s])
        c.bc_rho[s], c.bc_ux[s], c.bc_uy[s], c.bc_T[s] = float(bc_rho[s]), float(bc_ux[s]), float(bc_uy[s]), float(bc_T[s])
    return c


def _flatten(levels, depth):
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


class Grid:
    """One simulation: lbm_grid_create (host, no CUDA) [+ bind() to a torch-owned device arena and stream]."""

    def __init__(self, cfg, split=None, solid=None):
        self.cfg = cfg
        self.Q = cfg.lattice
        self.depth = cfg.depth
        so, sx = _flatten(split, cfg.depth)
        zo, zx = _flatten(solid, cfg.depth)
        h = C.c_void_p()
        self.h = None
        _check("lbm_grid_create", lib().lbm_grid_create(C.byref(cfg), _ptr(so), _ptr(sx), _ptr(zo), _ptr(zx), C.byref(h)))
        self.h = h
        self.info = LbmGridInfo()
        _check("lbm_grid_query", lib().lbm_grid_query(h, C.byref(self.info)))
        self.n = [int(self.info.n_cells[l]) for l in range(self.depth + 1)]
        self.off = np.concatenate([[0], np.cumsum(self.n)]).astype(np.int64)
        self.ntot = int(self.info.n_total)
        self.arena = None
        self.stream = None

    @classmethod
    def from_case(cls, case, precision=64, **device_options):
        """device_options: addressing=ADDR_*, no_pdl=0|1, pipeline=PIPE_*, pipe_max_ctas (lbm_config; they never change the result)."""
        kw = dict(case.model_kwargs(), **device_options)
        if precision == 32:      # Newton tolerance of single-precision runs (1e-12 in fp64, 1e-5 in fp32)
            kw["newton_tol"] = max(kw["newton_tol"], 1e-5)
        return cls(make_config(precision=precision, **kw), case.mesh.split, case.mesh.solid)

    def close(self):
        if getattr(self, "h", None):
            lib().lbm_destroy(self.h)
            self.h = None
        self.arena = None

    def __del__(self):
        self.close()

    # ---- host tables (bit-exact checks)
    def tau(self, l):
        return float(self.info.tau[l])

    def cells(self, l):
        n = self.n[l]
        ix = np.zeros(n, np.int32); iy = np.zeros(n, np.int32); ty = np.zeros(n, np.int32); aux = np.zeros(n, np.int32)
        _check("lbm_get_cells", lib().lbm_get_cells(self.h, l, _ptr(ix), _ptr(iy), _ptr(ty), _ptr(aux)))
        return ix, iy, ty, aux

    def nbr(self, l):
        a = np.zeros((self.n[l], self.Q - 1), np.int32)
        _check("lbm_get_nbr", lib().lbm_get_nbr(self.h, l, _ptr(a)))
        return a

    def sponge(self, l):
        a = np.zeros(self.n[l])
        _check("lbm_get_sponge", lib().lbm_get_sponge(self.h, l, _ptr(a)))
        return a

    def bricks(self, l):
        """(tiles9 [n_bricks, 9], table [Q-1, 64]) of lbm_get_bricks."""
        nb = int(self.info.n_bricks[l])
        t9 = np.zeros((nb, 9), np.int32); tab = np.zeros((self.Q - 1, 64), np.uint16)
        _check("lbm_get_bricks", lib().lbm_get_bricks(self.h, l, _ptr(t9) if nb else None, _ptr(tab)))
        return t9, tab

    def ghosts(self, l):
        ng = int(self.info.n_coarse_ghosts[l])
        co = np.zeros(ng, np.int32); ch = np.zeros((ng, 4), np.int32); m = np.zeros(ng, np.uint64)
        if ng:
            _check("lbm_get_ghosts", lib().lbm_get_ghosts(self.h, l, _ptr(co), _ptr(ch), _ptr(m)))
        return co, ch, m

    def schedule(self):
        n = lib().lbm_get_schedule(self.h, None, None, 0)
        k = np.zeros(n, np.int32); lv = np.zeros(n, np.int32)
        lib().lbm_get_schedule(self.h, _ptr(k), _ptr(lv), n)
        return k, lv

    # ---- device
    def bind(self, device="cuda:0", stream=None):
        """Allocates the device arena with torch and attaches it and torch's stream to the grid."""
        import torch
        if not torch.cuda.is_available():
            raise LbmError("lbm_grid_bind (no CUDA device; there is no CPU fallback)", ECUDA)
        dev = torch.device(device)
        self.arena = torch.empty(int(self.info.arena_bytes) + 256, dtype=torch.uint8, device=dev)
        base = self.arena.data_ptr()
        aligned = (base + 255) // 256 * 256
        with torch.cuda.device(dev):
            self.stream = stream if stream is not None else torch.cuda.Stream(device=dev)
            _check("lbm_grid_bind", lib().lbm_grid_bind(self.h, C.c_void_p(aligned), C.c_size_t(int(self.info.arena_bytes)),
                                                        C.c_void_p(self.stream.cuda_stream)))
        return self

    def init_fields(self, rho, ux, uy, T=None):
        a = [np.ascontiguousarray(x, dtype=np.float64) for x in (rho, ux, uy)]
        t = None if T is None else np.ascontiguousarray(T, dtype=np.float64)
        for x in a:
            assert x.size == self.ntot
        return lib().lbm_init_fields(self.h, _ptr(a[0]), _ptr(a[1]), _ptr(a[2]), _ptr(t))

    def step(self, n=1):
        _check("lbm_step", lib().lbm_step(self.h, int(n)))

    def step_fine(self, n=1):
        _check("lbm_step_fine", lib().lbm_step_fine(self.h, int(n)))

    def set_tau0(self, tau0):
        _check("lbm_set_relaxation", lib().lbm_set_relaxation(self.h, float(tau0)))

    def set_bc_state(self, side, rho, ux, uy, T=0.0):
        _check("lbm_set_boundary_state", lib().lbm_set_boundary_state(self.h, int(side), float(rho), float(ux), float(uy), float(T)))

    def transfer_from(self, src):
        """lbm_transfer: takes over the state of `src` (another tree over the same box) by copy / explosion / coalescence."""
        _check("lbm_transfer", lib().lbm_transfer(self.h, src.h))

    def sync(self):
        return lib().lbm_sync(self.h)

    def last_step_ms(self):
        ms = lib().lbm_last_step_ms(self.h)
        if ms < 0:
            raise LbmError("lbm_last_step_ms", int(ms))
        return ms

    def kernel_name(self):
        return lib().lbm_kernel_name(self.h).decode()

    def newton_iterations(self):
        """(Newton steps, equilibrium solves) counted on the device since bind (lbm_newton_iterations)."""
        it, ns = C.c_int64(0), C.c_int64(0)
        _check("lbm_newton_iterations", lib().lbm_newton_iterations(self.h, C.byref(it), C.byref(ns)))
        return it.value, ns.value

    def macroscopic(self, out=None):
        """rho, ux, uy, T of every stored cell; `out` = four caller-owned float64 arrays (e.g. pinned) to fill."""
        if out is not None:
            r, u, v, T = out
            for x in out:
                assert x.dtype == np.float64 and x.size == self.ntot and x.flags.c_contiguous
        else:
            r = np.zeros(self.ntot); u = np.zeros(self.ntot); v = np.zeros(self.ntot); T = np.zeros(self.ntot)
        _check("lbm_get_macroscopic", lib().lbm_get_macroscopic(self.h, _ptr(r), _ptr(u), _ptr(v), _ptr(T)))
        return r, u, v, T

    def macroscopic_at(self, l, cells):
        """rho, ux, uy, T of the given storage indices of level l (lbm_get_macroscopic_at)."""
        idx = np.ascontiguousarray(cells, dtype=np.int32)
        out = [np.zeros(idx.size) for _ in range(4)]
        _check("lbm_get_macroscopic_at", lib().lbm_get_macroscopic_at(self.h, int(l), int(idx.size), _ptr(idx), *[_ptr(o) for o in out]))
        return tuple(out)

    def sensor(self):
        """eps of Eq. 52 of the current state of every stored cell, flat over the levels (lbm_get_sensor)."""
        e = np.zeros(self.ntot)
        _check("lbm_get_sensor", lib().lbm_get_sensor(self.h, _ptr(e)))
        return e

    def macroscopic_at_static(self, l, cells):
        """The same through lbm_get_macroscopic_at_static: scratch in the library's static device array, no allocation,
        at most STATIC_PROBE_MAX cells per call."""
        idx = np.ascontiguousarray(cells, dtype=np.int32)
        out = [np.zeros(idx.size) for _ in range(4)]
        _check("lbm_get_macroscopic_at_static",
               lib().lbm_get_macroscopic_at_static(self.h, int(l), int(idx.size), _ptr(idx), *[_ptr(o) for o in out]))
        return tuple(out)

    def populations(self, l, which=0):
        cnt = 8 if which == 2 else self.Q
        a = np.zeros((self.n[l], cnt))
        _check("lbm_get_populations", lib().lbm_get_populations(self.h, l, which, _ptr(a)))
        return a

    def set_populations(self, l, which, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        _check("lbm_set_populations", lib().lbm_set_populations(self.h, l, which, _ptr(a)))
