"""Seeded, synthetic input generators shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic: it only produces mesh descriptions (which
quadtree cells are split, which positions are solid), model parameters and initial macroscopic
fields, shaped like the paper's workloads:

  tgv       config 1  uniform periodic box, Taylor-Green vortex          (textbook; BASELINE configs[0])
  cavity    config 2  lid-driven cavity, fine band along the walls       (paper Sec. 5.2)
  cylinder  config 3  flow past a cylinder, levels graded by distance    (paper Sec. 5.3 / Table 2)
  riemann   config 4  four-quadrant 2-D Riemann problem, uniform box     (paper Sec. 6.2)
  naca      config 5  NACA0012, levels graded by distance to the chord   (paper Sec. 6.3-6.4)

They stand in for the paper's benchmark cases; no external dataset or geometry file is used.
Numeric codes below are interface constants of the mesh/model description (the same values are
declared independently in include/lbm.h and oracle/oracle.h).
"""
from dataclasses import dataclass, field
import math

import numpy as np

# collision models / boundary kinds / cell types (interface constants)
BGK, RR, NUMEQ = 0, 1, 2
BC_PERIODIC, BC_WALL, BC_MOVING_WALL, BC_INFLOW_VBB, BC_DIRICHLET_EQ, BC_DIRICHLET_EQ_RHO_EXTRAP, BC_NEUMANN = range(7)
FLUID, FINE_GHOST, COARSE_GHOST, NEUMANN, DIRICHLET = range(5)

CS2 = {9: 1.0 / 3.0, 13: 0.5, 21: 2.0 / 3.0, 37: 0.697953322019683}   # Table 4 P:815 (used for Mach -> velocity only)
SOD_T0 = {13: 0.35, 21: 0.9, 37: 1.0}      # inviscid reference temperatures of the numerical equilibria


@dataclass
class Mesh:
    """Quadtree given by its internal nodes: split[l] = (n,2) int32 (ix,iy) of level-l cells that are
    split into four level-(l-1) cells; solid[l] = level-l positions that are solid. Level 0 = finest."""
    depth: int
    nx_coarse: int
    ny_coarse: int
    split: list
    solid: list


@dataclass
class Case:
    name: str
    mesh: Mesh
    lattice: int = 9
    collision: int = BGK
    ddf: int = 0
    sensor: int = 0
    trace_eq: int = 0
    tau0: float = 0.6
    T0: float = 0.0
    gamma: float = 1.4
    sensor_A: float = 1.5
    newton_tol: float = 1e-12
    newton_max_iter: int = 50
    bc: tuple = (0, 0, 0, 0)
    bc_rho: tuple = (1.0, 1.0, 1.0, 1.0)
    bc_ux: tuple = (0.0, 0.0, 0.0, 0.0)
    bc_uy: tuple = (0.0, 0.0, 0.0, 0.0)
    bc_T: tuple = (0.0, 0.0, 0.0, 0.0)
    sponge: object = None      # None or (x0, y0, r0, r1, sigma_max, rho_inf): pressure-relaxation sponge, Eq. 10-11
    fields: object = None      # callable(level, ix, iy) -> rho, ux, uy, T  (arrays; centres are (ix+.5)*2^level)
    meta: dict = field(default_factory=dict)

    def model_kwargs(self):
        return dict(lattice=self.lattice, collision=self.collision, ddf=self.ddf, sensor=self.sensor,
                    trace_eq=self.trace_eq, depth=self.mesh.depth, nx_coarse=self.mesh.nx_coarse,
                    ny_coarse=self.mesh.ny_coarse, tau0=self.tau0, T0=self.T0, gamma=self.gamma,
                    sensor_A=self.sensor_A, newton_tol=self.newton_tol, newton_max_iter=self.newton_max_iter,
                    bc=self.bc, bc_rho=self.bc_rho, bc_ux=self.bc_ux, bc_uy=self.bc_uy, bc_T=self.bc_T, sponge=self.sponge)


def empty_levels(depth):
    return [np.zeros((0, 2), np.int32) for _ in range(depth + 1)]


def uniform_mesh(nx, ny):
    return Mesh(0, nx, ny, empty_levels(0), empty_levels(0))


def build_mesh(depth, nx_coarse, ny_coarse, refine, solid=None):
    """Top-down refinement. refine(level, ix, iy) -> bool array (split this level-`level` cell, level >= 1);
    solid(level, ix, iy) -> bool array, evaluated on unsplit cells of every level."""
    split = empty_levels(depth)
    sol = empty_levels(depth)
    iy, ix = np.meshgrid(np.arange(ny_coarse, dtype=np.int32), np.arange(nx_coarse, dtype=np.int32), indexing="ij")
    ix = ix.ravel(); iy = iy.ravel()
    for l in range(depth, -1, -1):
        if l >= 1 and refine is not None:
            m = np.asarray(refine(l, ix, iy), dtype=bool)
        else:
            m = np.zeros(ix.shape, bool)
        split[l] = np.stack([ix[m], iy[m]], axis=1).astype(np.int32)
        lx, ly = ix[~m], iy[~m]
        if solid is not None and lx.size:
            s = np.asarray(solid(l, lx, ly), dtype=bool)
            sol[l] = np.stack([lx[s], ly[s]], axis=1).astype(np.int32)
        if l >= 1:
            px, py = ix[m], iy[m]
            ix = np.concatenate([2 * px, 2 * px + 1, 2 * px, 2 * px + 1]).astype(np.int32)
            iy = np.concatenate([2 * py, 2 * py, 2 * py + 1, 2 * py + 1]).astype(np.int32)
    return Mesh(depth, nx_coarse, ny_coarse, split, sol)


def centres(level, ix, iy):
    """Cell centres in finest-level lattice units (cell-centred grid)."""
    h = float(1 << level)
    return (np.asarray(ix, np.float64) + 0.5) * h, (np.asarray(iy, np.float64) + 0.5) * h


def hash_uniform(seed, level, ix, iy, stream):
    """Counter-based uniform numbers in [-1,1): splitmix64 of (seed, stream, level, ix, iy)."""
    with np.errstate(over="ignore"):
        z = (np.asarray(ix).astype(np.uint64) << np.uint64(32)) ^ (np.asarray(iy).astype(np.uint64) & np.uint64(0xFFFFFFFF))
        z = z + np.uint64((seed * 0x9E3779B97F4A7C15 + stream * 0xBF58476D1CE4E5B9 + level * 0x94D049BB133111EB) & 0xFFFFFFFFFFFFFFFF)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 / 9007199254740992.0) - 1.0


# ----------------------------------------------------------------------------- config 1
def tgv(n=64, u0=0.05, tau=0.6, lattice=9, collision=BGK, pressure_init=True):
    """Taylor-Green vortex on an n x n periodic box (BASELINE configs[0]; reading S21 for rho)."""
    k = 2.0 * math.pi / n
    cs2 = CS2[lattice]

    def fields(level, ix, iy):
        x, y = centres(level, ix, iy)
        ux = -u0 * np.cos(k * x) * np.sin(k * y)
        uy = u0 * np.sin(k * x) * np.cos(k * y)
        rho = 1.0 - (u0 * u0 / (4.0 * cs2)) * (np.cos(2 * k * x) + np.cos(2 * k * y)) if pressure_init else np.ones_like(x)
        return rho, ux, uy, np.full_like(x, cs2)

    return Case("tgv", uniform_mesh(n, n), lattice=lattice, collision=collision, tau0=tau, fields=fields,
                meta=dict(n=n, u0=u0, k=k, nu=cs2 * (tau - 0.5)))


# ----------------------------------------------------------------------------- config 2
def cavity(scale=1.0, collision=RR, re=1000.0, u_lid=0.1, trace_eq=0, lattice=9):
    """Lid-driven cavity: coarse N x N (N = 128*scale), level-1 cells split iff within 16*scale coarse
    cells of a wall; finest-equivalent 2N x 2N; bounce-back walls, moving lid on top (side 3)."""
    N = int(round(128 * scale)); band = int(round(16 * scale))

    def refine(level, ix, iy):
        return (ix < band) | (ix >= N - band) | (iy < band) | (iy >= N - band)

    mesh = build_mesh(1, N, N, refine)
    nu0 = u_lid * (2 * N) / re
    tau0 = 0.5 + nu0 / CS2[lattice]

    def fields(level, ix, iy):
        o = np.ones(len(ix))
        return o, 0 * o, 0 * o, CS2[lattice] * o

    return Case("cavity", mesh, lattice=lattice, collision=collision, trace_eq=trace_eq, tau0=tau0,
                bc=(BC_WALL, BC_WALL, BC_WALL, BC_MOVING_WALL), bc_ux=(0, 0, 0, u_lid), fields=fields,
                meta=dict(N=N, band=band, re=re, u_lid=u_lid, nu0=nu0))


def cavity_uniform(n=256, collision=RR, re=1000.0, u_lid=0.1, lattice=9, inflow=0.0):
    """Lid-driven cavity on a uniform n x n box (the paper's uniform Cartesian benchmark): bounce-back walls, moving
    lid on top; inflow > 0 adds a wall-normal velocity on the left side (velocity bounce-back with mass flux, tests)."""
    nu0 = u_lid * n / re
    tau0 = 0.5 + nu0 / CS2[lattice]

    def fields(level, ix, iy):
        o = np.ones(len(ix))
        return o, 0 * o, 0 * o, CS2[lattice] * o

    left = BC_INFLOW_VBB if inflow else BC_WALL
    return Case("cavity_uniform", uniform_mesh(n, n), lattice=lattice, collision=collision, tau0=tau0,
                bc=(left, BC_WALL, BC_WALL, BC_MOVING_WALL), bc_ux=(inflow, 0, 0, u_lid), fields=fields,
                meta=dict(N=n, re=re, u_lid=u_lid, nu0=nu0))


# ----------------------------------------------------------------------------- config 3
CYL_RADII_D = (6.5, 11.0, 17.0, 23.0, 29.0)   # refinement radii R_0..R_4 in cylinder diameters


def cylinder(D=200, depth=5, mach=0.2, re=150.0, seed=1234, collision=RR, lattice=9, radii=CYL_RADII_D, sponge_d=None):
    """Flow past a circular cylinder of diameter D finest cells in a 64D x 64D box, `depth`+1 levels graded
    by distance from the cylinder; left inflow (velocity bounce-back), other sides Neumann.
    sponge_d = (r0, r1, sigma_max) in diameters switches the pressure-relaxation sponge of Eq. 10-11 on around the
    cylinder centre with rho_inf = 1 (the paper: 130 D, 180 D, 0.1 in a 400 D domain; here e.g. (24, 30, 0.1))."""
    L = 64 * D
    nc = L >> depth
    assert nc << depth == L, "64*D must be divisible by 2^depth"
    cxc = cyc = L / 2.0
    cs2 = CS2[lattice]
    u_inf = mach * math.sqrt(cs2)

    def refine(level, ix, iy):
        x, y = centres(level, ix, iy)
        R = radii[level - 1] * D
        return (x - cxc) ** 2 + (y - cyc) ** 2 < R * R

    def solid(level, ix, iy):
        if level != 0:
            return np.zeros(len(ix), bool)
        x, y = centres(level, ix, iy)
        return (x - cxc) ** 2 + (y - cyc) ** 2 < (0.5 * D) ** 2

    mesh = build_mesh(depth, nc, nc, refine, solid)
    nu0 = u_inf * D / re
    tau0 = 0.5 + nu0 / cs2

    def fields(level, ix, iy):
        o = np.ones(len(ix))
        ux = u_inf * (1.0 + 1e-4 * hash_uniform(seed, level, ix, iy, 0))
        uy = u_inf * 1e-4 * hash_uniform(seed, level, ix, iy, 1)
        return o, ux, uy, cs2 * o

    sponge = None if sponge_d is None else (cxc, cyc, sponge_d[0] * D, sponge_d[1] * D, sponge_d[2], 1.0)
    return Case("cylinder", mesh, lattice=lattice, collision=collision, tau0=tau0, sponge=sponge,
                bc=(BC_INFLOW_VBB, BC_NEUMANN, BC_NEUMANN, BC_NEUMANN), bc_ux=(u_inf, 0, 0, 0), fields=fields,
                meta=dict(D=D, u_inf=u_inf, re=re, nu0=nu0, mach=mach))


# ----------------------------------------------------------------------------- config 4
def riemann(n=2048, seed=7, lattice=37, periodic=False, sensor=1, tau0=0.5, gamma=1.4, sensor_A=1.5, collision=BGK, T0=None,
            mach_max=1.5):
    """Four-quadrant 2-D Riemann problem on a uniform n x n box. Quadrant states are drawn from a seeded
    generator: rho in [0.5, 8], T/T0 in [0.7, 1.4], |u|/sqrt(gamma T) <= mach_max, |u| < 1.9 (reading S17).
    collision=BGK: the thermal polynomial model of BASELINE configs[3] (T0 = c_s^2); collision=NUMEQ: the numerical
    equilibrium the paper itself runs on this lattice, reference temperature T0 (default: the inviscid value of
    P:369)."""
    rng = np.random.RandomState(seed)
    Tref = CS2[lattice] if collision != NUMEQ else (SOD_T0[lattice] if T0 is None else T0)
    rho_q = np.exp(rng.uniform(math.log(0.5), math.log(8.0), 4))
    T_q = Tref * rng.uniform(0.7, 1.4, 4)
    ma_q = rng.uniform(0.0, 1.5, 4) * (mach_max / 1.5)
    ang = rng.uniform(0.0, 2 * math.pi, 4)
    sp = np.minimum(ma_q * np.sqrt(gamma * T_q), 1.9)
    ux_q = sp * np.cos(ang); uy_q = sp * np.sin(ang)

    def fields(level, ix, iy):
        q = (np.asarray(ix) >= n // 2).astype(np.int64) + 2 * (np.asarray(iy) >= n // 2).astype(np.int64)
        return rho_q[q], ux_q[q], uy_q[q], T_q[q]

    kind = BC_PERIODIC if periodic else BC_NEUMANN
    return Case("riemann", uniform_mesh(n, n), lattice=lattice, collision=collision, ddf=1, sensor=sensor, tau0=tau0,
                T0=(Tref if collision == NUMEQ else 0.0), gamma=gamma, sensor_A=sensor_A, bc=(kind,) * 4, fields=fields,
                meta=dict(n=n, rho=rho_q, T=T_q, ux=ux_q, uy=uy_q))


# ----------------------------------------------------------------------------- Sod shock tube
def sod(L=8192, lattice=21, mesh="unif", periodic=True, sensor_A=1.5, gamma=1.4, ny=None):
    """Inviscid Sod shock tube (Eq. 12: (p, rho, u) = (10, 8, 0) p0, rho0 left of x = L/2, (1, 1, 0) right) on an
    L x L box (L = finest-equivalent cells per side) with numerical equilibria + g + sensor (A = 1.5), tau = 1/2
    (P:940).  Meshes of Sec. 6.1 / Table 3: unif; hori (fine below y = L/2), band (fine for
    L/4 <= x < 3L/4), sqr (fine L/2 square at the centre), each two levels over a coarse L/2 x L/2 box.
    periodic=True (throughput runs): fully periodic box, i.e. a second, mirrored Riemann problem at the seam x = 0;
    periodic=False (physics pin, unif only): Neumann ends in x, periodic in y; ny: height of the unif box (default L)."""
    T0 = SOD_T0[lattice]
    rho_r, T_r = 1.0, T0                     # right state: rho0 = 1, p0 = rho0 T0
    rho_l, T_l = 8.0, 10.0 / 8.0 * T0        # p = 10 p0, rho = 8 rho0

    def fields(level, ix, iy):
        x, _ = centres(level, ix, iy)
        left = x < 0.5 * L
        z = np.zeros(len(x))
        return np.where(left, rho_l, rho_r), z, z, np.where(left, T_l, T_r)

    if mesh == "unif":
        m = uniform_mesh(L, L if ny is None else ny)
    else:
        nc = L // 2
        assert 2 * nc == L and mesh in ("hori", "band", "sqr"), mesh

        def refine(level, ix, iy):
            inx = (ix >= nc // 4) & (ix < 3 * nc // 4)
            iny = (iy >= nc // 4) & (iy < 3 * nc // 4)
            return {"hori": iy < nc // 2, "band": inx, "sqr": inx & iny}[mesh]
        m = build_mesh(1, nc, nc, refine)
    bc = (BC_PERIODIC,) * 4 if periodic else (BC_NEUMANN, BC_NEUMANN, BC_PERIODIC, BC_PERIODIC)
    return Case("sod", m, lattice=lattice, collision=NUMEQ, ddf=1, sensor=1, tau0=0.5, T0=T0, gamma=gamma, sensor_A=sensor_A,
                bc=bc, fields=fields, meta=dict(L=L, mesh=mesh, left=(rho_l, 0.0, T_l), right=(rho_r, 0.0, T_r)))


# ----------------------------------------------------------------------------- config 5
NACA_RADII_C = (1.0, 2.25, 5.0, 9.0, 12.5, 14.0)   # R_0..R_5 in chords


def naca_thickness(xc, t=0.12):
    """Closed-form NACA 4-digit half thickness at chord fraction xc in [0,1]."""
    xc = np.clip(xc, 0.0, 1.0)
    return 5.0 * t * (0.2969 * np.sqrt(xc) - 0.1260 * xc - 0.3516 * xc ** 2 + 0.2843 * xc ** 3 - 0.1015 * xc ** 4)


def naca(chord=1024, depth=6, mach=0.8, aoa_deg=0.0, re=1e4, lattice=21, T0=0.65, gamma=1.4, sensor_A=1.35,
         radii=NACA_RADII_C, collision=NUMEQ):
    """NACA0012 of `chord` finest cells centred in a 30C x 30C box; levels graded by distance to the chord
    segment; left/top/bottom equilibrium Dirichlet, right Neumann."""
    L = 30 * chord
    nc = L >> depth
    assert nc << depth == L, "30*chord must be divisible by 2^depth"
    x0 = y0 = L / 2.0
    a = math.radians(aoa_deg)
    ca, sa = math.cos(a), math.sin(a)

    def frame(level, ix, iy):
        x, y = centres(level, ix, iy)
        x = x - x0; y = y - y0
        return ca * x - sa * y, sa * x + ca * y      # airfoil frame, chord on [-C/2, C/2] x {0}

    def refine(level, ix, iy):
        xa, ya = frame(level, ix, iy)
        dx = np.maximum(np.abs(xa) - 0.5 * chord, 0.0)
        R = radii[level - 1] * chord
        return dx * dx + ya * ya < R * R

    def solid(level, ix, iy):
        if level != 0:
            return np.zeros(len(ix), bool)
        xa, ya = frame(level, ix, iy)
        xc = xa / chord + 0.5
        return (xc >= 0.0) & (xc <= 1.0) & (np.abs(ya) < chord * naca_thickness(xc))

    mesh = build_mesh(depth, nc, nc, refine, solid)
    u_inf = mach * math.sqrt(gamma * T0)
    nu0 = u_inf * chord / re
    tau0 = 0.5 + nu0 / T0
    far = BC_DIRICHLET_EQ if mach >= 1.0 else BC_DIRICHLET_EQ_RHO_EXTRAP

    def fields(level, ix, iy):
        o = np.ones(len(ix))
        return o, u_inf * o, 0 * o, T0 * o

    return Case("naca", mesh, lattice=lattice, collision=collision, ddf=1, sensor=1, tau0=tau0, T0=T0, gamma=gamma,
                sensor_A=sensor_A, bc=(far, BC_NEUMANN, far, far), bc_rho=(1, 1, 1, 1), bc_ux=(u_inf,) * 4,
                bc_uy=(0,) * 4, bc_T=(T0,) * 4, fields=fields,
                meta=dict(chord=chord, u_inf=u_inf, mach=mach, aoa=aoa_deg, nu0=nu0))


# ----------------------------------------------------------------------------- helpers
def patch(nc=32, lo=8, hi=24, depth=1, lattice=9, collision=BGK, tau0=0.8, periodic=True, fields=None, **kw):
    """Periodic (or walled) box of nc x nc coarse cells with a refined square patch [lo,hi)^2 (tests)."""
    def refine(level, ix, iy):
        if level != depth:
            # nested patches: shrink by a margin on finer levels
            s = 1 << (depth - level)
            m = 6 * s * (depth - level)
            return (ix >= lo * s + m) & (ix < hi * s - m) & (iy >= lo * s + m) & (iy < hi * s - m)
        return (ix >= lo) & (ix < hi) & (iy >= lo) & (iy < hi)

    mesh = build_mesh(depth, nc, nc, refine)
    kind = BC_PERIODIC if periodic else BC_WALL
    return Case("patch", mesh, lattice=lattice, collision=collision, tau0=tau0, bc=(kind,) * 4, fields=fields, **kw)


def stripe(nc=32, lo=8, hi=24, lattice=9, collision=BGK, tau0=0.8, fields=None, **kw):
    """Periodic box with a refined vertical stripe lo <= ix < hi: two straight interfaces (tests, pin P8)."""
    def refine(level, ix, iy):
        return (ix >= lo) & (ix < hi)

    mesh = build_mesh(1, nc, nc, refine)
    return Case("stripe", mesh, lattice=lattice, collision=collision, tau0=tau0, bc=(BC_PERIODIC,) * 4, fields=fields, **kw)


# ----------------------------------------------------------------------------- start-up ramps
def viscosity_ramp_tau0(tau0, step, nsteps, factor=100.0):
    """tau_0 at coarse step `step` of the viscosity ramp: nu starts at factor * nu and decreases linearly to nu over
    nsteps steps; tau - 1/2 is proportional to nu on every level (Eq. 3), so the ramp scales tau_0 - 1/2."""
    m = factor - (factor - 1.0) * min(step / float(nsteps), 1.0)
    return 0.5 + (tau0 - 0.5) * m


def mach_ramp_factor(step, nsteps, start=0.5):
    """Fraction of the nominal boundary velocity imposed at coarse step `step` of the Mach ramp (the free-stream Mach
    number starts below the target and is raised to it over one convective time)."""
    return start + (1.0 - start) * min(step / float(nsteps), 1.0)


def eval_fields(case, levels_ix_iy):
    """levels_ix_iy: list over levels 0..depth of (ix, iy) arrays in storage order -> flat rho, ux, uy, T."""
    out = [[], [], [], []]
    for l, (ix, iy) in enumerate(levels_ix_iy):
        r = case.fields(l, ix, iy)
        for k in range(4):
            out[k].append(np.broadcast_to(np.asarray(r[k], np.float64), (len(ix),)).copy())
    return tuple(np.concatenate(o) if o else np.zeros(0) for o in out)
