"""Pins for the oracle's boundary cells and links that no other pin reaches (pins P13-P16):
equilibrium Dirichlet cells and their density extrapolation, Neumann replica cells (reading S13), the W
boundary layers ("as many layers as the lattice size"), the equilibrated trace of the recursive-regularised
collision (reading S7) and velocity bounce-back with a NORMAL wall velocity (the inflow of the Aeolian
cylinder).  Each test derives its expectation from the paper's statement with its own arithmetic (clamped
coordinates, closed-form equilibria, moment constraints, the lattice flux sum) -- never from the oracle's update."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2504_04465_b200 import workloads as W
from helpers import oracle_from_case

REACH = {9: 1, 13: 2, 21: 3, 37: 3}                     # "lattice size" of Table 4


def box_case(nx, ny, bc, fields, lattice=9, collision=W.BGK, ddf=0, sensor=0, tau0=0.8, T0=0.0, **kw):
    return W.Case("box", W.uniform_mesh(nx, ny), lattice=lattice, collision=collision, ddf=ddf, sensor=sensor, tau0=tau0,
                  T0=T0, bc=bc, fields=fields, **kw)


def clamp_source(ix, iy, nx, ny):
    """Nearest in-box cell along the boundary normal (diagonal at corners): P:938 'nearest fluid cell'."""
    return np.clip(ix, 0, nx - 1), np.clip(iy, 0, ny - 1)


def side_of(ix, iy, nx, ny):
    """Side a boundary cell belongs to; a corner cell (outside in x and y) takes the y side."""
    ox = np.where(ix < 0, 0, np.where(ix >= nx, 1, -1))
    oy = np.where(iy < 0, 2, np.where(iy >= ny, 3, -1))
    return np.where(oy >= 0, oy, ox)


def index_of(ix, iy):
    return {(int(x), int(y)): c for c, (x, y) in enumerate(zip(ix, iy))}


def feq_product_d2q9(rho, ux, uy, cx, cy):
    """Closed form of the extended D2Q9 equilibrium (product form; pin P2 checks the oracle's polynomial against it)."""
    def phi(c, u):
        return np.where(c == 0, 2.0 / 3.0 - u * u, (1.0 + 3.0 * c * u + 3.0 * u * u) / 6.0)
    return rho * phi(cx, ux) * phi(cy, uy)


def pulse_fields(nx, ny, u=(0.08, 0.03), T0=1.0 / 3.0, amp=0.05):
    """A Gaussian density (and temperature) pulse close to the right / top sides, carried by a uniform flow."""
    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        r2 = (x - 0.8 * nx) ** 2 + (y - 0.7 * ny) ** 2
        bump = amp * np.exp(-r2 / (0.02 * nx * ny))
        o = np.ones(len(x))
        return 1.0 + bump, u[0] * o, u[1] * o, T0 * (1.0 + 0.5 * bump)
    return fields


# ----------------------------------------------------------------------------- P13: boundary layers
@pytest.mark.parametrize("Q", [9, 13, 21, 37])
@pytest.mark.parametrize("kind", [W.BC_NEUMANN, W.BC_DIRICHLET_EQ])
def test_boundary_layers_are_as_wide_as_the_lattice(Q, kind):
    """'As many layers as the lattice size': a box with four boundary-cell sides stores exactly the frame of width
    W = 1, 2, 3, 3 (D2Q9/13/21/37) around it, corners included, after the in-box cells, ordered by (iy, ix); every link
    of every in-box cell then finds a stored cell, and aux points to the clamped source."""
    nx, ny, Wd = 12, 9, REACH[Q]
    case = box_case(nx, ny, (kind,) * 4, pulse_fields(nx, ny), lattice=Q)
    g = oracle_from_case(case, init=False)
    ix, iy, ty, aux = g.cells(0)
    inbox = (ix >= 0) & (ix < nx) & (iy >= 0) & (iy < ny)
    assert inbox[:nx * ny].all() and not inbox[nx * ny:].any()
    frame = {(x, y) for y in range(-Wd, ny + Wd) for x in range(-Wd, nx + Wd) if not (0 <= x < nx and 0 <= y < ny)}
    got = list(zip(ix[nx * ny:].tolist(), iy[nx * ny:].tolist()))
    assert set(got) == frame and len(got) == len(frame) == (nx + 2 * Wd) * (ny + 2 * Wd) - nx * ny
    assert got == sorted(got, key=lambda p: (p[1], p[0]))
    assert (ty[nx * ny:] == (O.NEUMANN if kind == W.BC_NEUMANN else O.DIRICHLET)).all()
    where = index_of(ix, iy)
    sx, sy = clamp_source(ix[nx * ny:], iy[nx * ny:], nx, ny)
    assert aux[nx * ny:].tolist() == [where[(int(a), int(b))] for a, b in zip(sx, sy)]
    cx, cy, w, opp, cs2, reach = O.lattice(Q)
    assert reach == Wd
    nb = g.nbr(0)
    for c in range(nx * ny):
        for i in range(1, Q):
            assert nb[c, i - 1] == where[(int(ix[c] - cx[i]), int(iy[c] - cy[i]))]


# ----------------------------------------------------------------------------- P13: equilibrium Dirichlet cells
DIRICHLET_MODELS = [(9, W.BGK, 0, 0.0), (9, W.RR, 0, 0.0), (21, W.NUMEQ, 1, 0.65)]


@pytest.mark.parametrize("Q,coll,ddf,T0", DIRICHLET_MODELS)
@pytest.mark.parametrize("kind", [W.BC_DIRICHLET_EQ, W.BC_DIRICHLET_EQ_RHO_EXTRAP])
def test_dirichlet_sides_keep_a_uniform_free_stream(Q, coll, ddf, T0, kind):
    """A uniform state equal to the imposed far-field state is a fixed point of the whole update with equilibrium
    Dirichlet sides of either kind (and a Neumann outflow on the right, the NACA set-up of P:418): rho, u, T stay
    uniform to rounding for 50 steps."""
    nx, ny = 14, 11
    Tb = T0 if coll == W.NUMEQ else 1.0 / 3.0
    rho0, u0, v0 = 1.1, 0.12, -0.04

    def fields(level, ix, iy):
        o = np.ones(len(ix))
        return rho0 * o, u0 * o, v0 * o, Tb * o
    case = box_case(nx, ny, (kind, W.BC_NEUMANN, kind, kind), fields, lattice=Q, collision=coll, ddf=ddf, sensor=ddf, T0=T0,
                    bc_rho=(rho0,) * 4, bc_ux=(u0,) * 4, bc_uy=(v0,) * 4, bc_T=(Tb,) * 4)
    g = oracle_from_case(case)
    assert g.step(50) == 0
    r, u, v, T = g.macroscopic()
    assert np.abs(r - rho0).max() < 1e-12 and np.abs(u - u0).max() < 1e-12 and np.abs(v - v0).max() < 1e-12
    if ddf:
        assert np.abs(T - Tb).max() < 1e-12


def _numeq_constraints(f, gpop, rho, ux, uy, T, cx, cy, gamma):
    """Worst violation of the eight moment constraints of Eq. 42-49 (2E = u^2 + 2T), of the exponential form of Eq. 39
    (ln f_i in the span of the eight monomials) and of g = (2 C_v - D) T f (Eq. 50): together they fix f^eq, g^eq uniquely."""
    r2 = cx * cx + cy * cy
    M = np.stack([np.ones(len(cx)), cx, cy, cx * cx, cx * cy, cy * cy, cx * r2, cy * r2], axis=1).astype(float)
    u2 = ux * ux + uy * uy
    m = rho * np.array([1.0, ux, uy, ux * ux + T, ux * uy, uy * uy + T, ux * (u2 + 4 * T), uy * (u2 + 4 * T)])
    e_mom = np.abs(f @ M - m).max()
    coef, res, rank, sv = np.linalg.lstsq(M, np.log(f), rcond=None)
    e_exp = np.abs(M @ coef - np.log(f)).max()
    e_g = np.abs(gpop - (2.0 / (gamma - 1.0) - 2.0) * T * f).max()
    return max(e_mom, e_exp, e_g)


@pytest.mark.parametrize("Q,coll,ddf,T0", DIRICHLET_MODELS)
@pytest.mark.parametrize("kind", [W.BC_DIRICHLET_EQ, W.BC_DIRICHLET_EQ_RHO_EXTRAP])
def test_dirichlet_cells_hold_the_equilibrium_of_the_imposed_state(Q, coll, ddf, T0, kind):
    """After one step on a NON-uniform field with a different state imposed on every side, every Dirichlet cell holds
    f^eq, g^eq of (rho_b, u_side, T_side): side = the y side at corners; rho_b = the side's imposed density, or
    (RHO_EXTRAP) the density of the nearest in-box cell along the normal, summed by the test from that cell's PRE-step
    populations.  D2Q9: compared with the closed product form; D2Q21 numerical equilibria: with the constraints of
    Eq. 39, 42-49, 50 that define them."""
    nx, ny, Wd = 13, 10, REACH[Q]
    Tb = T0 if coll == W.NUMEQ else 1.0 / 3.0
    bc_rho = (1.05, 0.9, 1.2, 0.95)
    bc_ux = (0.10, -0.03, 0.06, 0.02)
    bc_uy = (-0.02, 0.04, 0.05, -0.07)
    bc_T = tuple(Tb * s for s in (1.0, 1.1, 0.9, 1.05)) if ddf else (Tb,) * 4
    case = box_case(nx, ny, (kind,) * 4, pulse_fields(nx, ny, T0=Tb), lattice=Q, collision=coll, ddf=ddf, sensor=ddf, T0=T0,
                    bc_rho=bc_rho, bc_ux=bc_ux, bc_uy=bc_uy, bc_T=bc_T)
    g = oracle_from_case(case)
    assert g.step(2) == 0                                   # the in-box field next to the sides is no longer the initial one
    ix, iy, ty, aux = g.cells(0)
    where = index_of(ix, iy)
    cx, cy, w, opp, cs2, reach = O.lattice(Q)
    f_old = g.populations(0, 0).copy()
    assert g.step(1) == 0
    f_new = g.populations(0, 0)
    g_new = g.populations(0, 1) if ddf else None
    bcells = np.flatnonzero(ty == O.DIRICHLET)
    assert bcells.size == (nx + 2 * Wd) * (ny + 2 * Wd) - nx * ny
    sides = side_of(ix[bcells], iy[bcells], nx, ny)
    sx, sy = clamp_source(ix[bcells], iy[bcells], nx, ny)
    assert len(set(sides.tolist())) == 4
    worst = 0.0
    for b, sd, a, c in zip(bcells, sides, sx, sy):
        rho_b = bc_rho[sd] if kind == W.BC_DIRICHLET_EQ else f_old[where[(int(a), int(c))]].sum()
        if coll == W.NUMEQ:
            worst = max(worst, _numeq_constraints(f_new[b], g_new[b], rho_b, bc_ux[sd], bc_uy[sd], bc_T[sd], cx, cy, 1.4))
        else:
            worst = max(worst, np.abs(f_new[b] - feq_product_d2q9(rho_b, bc_ux[sd], bc_uy[sd], cx, cy)).max())
    assert worst < (5e-12 if coll == W.NUMEQ else 1e-15), worst
    if kind == W.BC_DIRICHLET_EQ_RHO_EXTRAP:
        # the extrapolated density really differs from cell to cell (the pulse sits next to the right / top sides)
        rho_b = np.array([f_old[where[(int(a), int(c))]].sum() for a, c in zip(sx, sy)])
        assert rho_b.max() - rho_b.min() > 1e-3


# ----------------------------------------------------------------------------- P14: Neumann replica cells
@pytest.mark.parametrize("Q,coll,ddf,T0", [(9, W.RR, 0, 0.0), (13, W.BGK, 0, 0.0), (21, W.NUMEQ, 1, 0.65), (37, W.BGK, 1, 0.0)])
def test_neumann_cells_copy_the_nearest_interior_cell(Q, coll, ddf, T0):
    """'Copy all populations from the nearest fluid cell': while a pulse leaves through the right / top sides,
    after every step each Neumann cell holds exactly the populations (f, g, lambda) of the in-box cell with clamped
    coordinates -- W layers deep, corners diagonal -- and the field next to the sides is not uniform."""
    nx, ny, Wd = 16, 12, REACH[Q]
    Tb = T0 if coll == W.NUMEQ else W.CS2[Q]
    case = box_case(nx, ny, (W.BC_NEUMANN,) * 4, pulse_fields(nx, ny, T0=Tb), lattice=Q, collision=coll, ddf=ddf, sensor=ddf,
                    T0=T0, tau0=0.7)
    g = oracle_from_case(case)
    ix, iy, ty, aux = g.cells(0)
    where = index_of(ix, iy)
    b = np.flatnonzero(ty == O.NEUMANN)
    assert b.size == (nx + 2 * Wd) * (ny + 2 * Wd) - nx * ny
    sx, sy = clamp_source(ix[b], iy[b], nx, ny)
    src = np.array([where[(int(a), int(c))] for a, c in zip(sx, sy)])
    which = [0] + ([1] if ddf else []) + ([2] if coll == W.NUMEQ else [])
    spread = 0.0
    for step in range(6):
        assert g.step(1) == 0
        for wsel in which:
            S = g.populations(0, wsel)
            assert np.array_equal(S[b], S[src]), (step, wsel)
        spread = max(spread, float(np.ptp(g.populations(0, 0)[src].sum(axis=1))))
    assert spread > 1e-3


@pytest.mark.parametrize("Q,coll", [(9, W.RR), (21, W.BGK)])
def test_neumann_sides_let_a_uniform_flow_through_unchanged(Q, coll):
    """Zero gradient: a uniform flow enters and leaves a box with four Neumann sides unchanged for 50 steps."""
    nx, ny = 12, 12

    def fields(level, ix, iy):
        o = np.ones(len(ix))
        return 0.9 * o, 0.1 * o, 0.05 * o, W.CS2[Q] * o
    g = oracle_from_case(box_case(nx, ny, (W.BC_NEUMANN,) * 4, fields, lattice=Q, collision=coll))
    f0 = g.populations(0, 0).copy()
    assert g.step(50) == 0
    assert np.abs(g.populations(0, 0) - f0).max() < 1e-14


def test_neumann_outflow_differs_from_a_periodic_or_mirrored_copy():
    """The pin above would also pass if the field at the sides were uniform; here the pulse reaches the right side and
    the Neumann layer is compared with the two plausible WRONG sources (periodic image, mirror image): it equals neither."""
    nx, ny = 16, 12
    g = oracle_from_case(box_case(nx, ny, (W.BC_NEUMANN,) * 4, pulse_fields(nx, ny), collision=W.RR, tau0=0.7))
    g.step(4)
    ix, iy, ty, aux = g.cells(0)
    where = index_of(ix, iy)
    f = g.populations(0, 0)
    right = [c for c in np.flatnonzero(ty == O.NEUMANN) if ix[c] == nx and 0 <= iy[c] < ny]
    assert len(right) == ny
    d_per = max(np.abs(f[c] - f[where[(0, int(iy[c]))]]).max() for c in right)
    assert d_per > 1e-4
    assert all(np.array_equal(f[c], f[where[(nx - 1, int(iy[c]))]]) for c in right)


# ----------------------------------------------------------------------------- P15: equilibrated trace
def _second_moments(f, cx, cy, cs2):
    rho = f.sum()
    ux, uy = (f * cx).sum() / rho, (f * cy).sum() / rho
    pxx = (f * cx * cx).sum() - rho * cs2 - rho * ux * ux
    pxy = (f * cx * cy).sum() - rho * ux * uy
    pyy = (f * cy * cy).sum() - rho * cs2 - rho * uy * uy
    return rho, ux, uy, pxx, pxy, pyy


@pytest.mark.parametrize("Q", [9, 13, 21])
def test_trace_eq_relaxes_the_trace_fully_and_the_deviator_with_tau(Q):
    """'Equilibrating the trace of second-order moments': with trace_eq the post-collision non-equilibrium
    stress Pi* = sum xi xi f* - rho c_s^2 I - rho u u has zero trace, while its deviatoric part (Pi_xx - Pi_yy, Pi_xy) is
    the pre-collision one times (1 - 1/tau); without trace_eq the trace is scaled by (1 - 1/tau) like the rest.  Moments
    are formed by the test from the populations (exact on the rational-weight lattices)."""
    cx, cy, w, opp, cs2, reach = O.lattice(Q)
    rng = np.random.RandomState(5 + Q)
    tau = 0.83
    keep = 1.0 - 1.0 / tau
    for trial in range(20):
        f = O.feq_poly(Q, 1.0 + 0.2 * rng.rand(), 0.1 * rng.randn(), 0.1 * rng.randn()) * (1.0 + 0.05 * rng.randn(Q))
        rho, ux, uy, pxx, pxy, pyy = _second_moments(f, cx, cy, cs2)
        assert abs(pxx + pyy) > 1e-4                                           # the input does carry a trace
        out = {}
        for te in (0, 1):
            cfg = O.make_config(lattice=Q, collision=O.RR, trace_eq=te, tau0=tau)
            fo, _, _, it = O.collide_cell(cfg, tau, f)
            out[te] = _second_moments(fo, cx, cy, cs2)
            assert abs(out[te][0] - rho) < 1e-14 and abs(out[te][1] - ux) < 1e-14 and abs(out[te][2] - uy) < 1e-14
        _, _, _, qxx, qxy, qyy = out[1]
        assert abs(qxx + qyy) < 1e-15
        assert abs((qxx - qyy) - keep * (pxx - pyy)) < 1e-15 and abs(qxy - keep * pxy) < 1e-15
        _, _, _, rxx, rxy, ryy = out[0]
        assert abs((rxx + ryy) - keep * (pxx + pyy)) < 1e-15
        assert abs((rxx - ryy) - keep * (pxx - pyy)) < 1e-15 and abs(rxy - keep * pxy) < 1e-15


@pytest.mark.parametrize("Q", [9, 13, 21, 37])
def test_trace_eq_is_a_no_op_on_a_traceless_stress(Q):
    """A non-equilibrium part made of the second-order Hermite polynomials H_xx - H_yy and H_xy only (no density, no
    momentum, no trace) is collided identically with and without trace_eq."""
    cx, cy, w, opp, cs2, reach = O.lattice(Q)
    rng = np.random.RandomState(11 + Q)
    for trial in range(10):
        feq = O.feq_poly(Q, 1.1, 0.07, -0.04)
        a, b = 0.02 * rng.randn(2)
        f = feq + w * (a * ((cx * cx - cs2) - (cy * cy - cs2)) + b * cx * cy)
        fo = [O.collide_cell(O.make_config(lattice=Q, collision=O.RR, trace_eq=te, tau0=0.7), 0.7, f)[0] for te in (0, 1)]
        assert np.abs(fo[0] - fo[1]).max() < 2e-16
        assert np.abs(fo[0] - feq).max() > 1e-4


# ----------------------------------------------------------------------------- P16: velocity bounce-back, normal velocity
@pytest.mark.parametrize("Q", [9, 13, 21])
def test_normal_inflow_injects_the_mass_flux_rho_u(Q):
    """Ladd's velocity bounce-back with a wall velocity NORMAL to the wall (the inflow of the cylinder case): a
    link crossing the inflow plane adds 2 w_i rho_w (xi_i . u_w) / c_s^2 to the reflected population, so the mass
    entering a channel closed by a wall at the other end is, per step, the sum of that term over the crossing links --
    for a uniform density rho u_in per unit height, since sum_{xi_x>0} 2 w_i xi_x^2 = c_s^2.  The density at the inlet is
    made non-uniform, the expected gain is summed by the test from the PRE-step populations, step by step."""
    nx, ny, u_in = 10, 8, 0.06
    cx, cy, w, opp, cs2, reach = O.lattice(Q)
    assert abs(sum(2 * w[i] * cx[i] * cx[i] for i in range(Q) if cx[i] > 0) - cs2) < 1e-15

    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        return 1.0 + 0.1 * np.sin(2 * math.pi * y / ny) * np.exp(-x / 3.0), 0.02 * np.ones(len(x)), np.zeros(len(x)), np.full(len(x), cs2)
    case = box_case(nx, ny, (W.BC_INFLOW_VBB, W.BC_WALL, W.BC_PERIODIC, W.BC_PERIODIC), fields, lattice=Q, collision=W.RR,
                    tau0=0.8, bc_ux=(u_in, 0, 0, 0))
    g = oracle_from_case(case)
    ix, iy, ty, aux = g.cells(0)
    nb = g.nbr(0)
    # links whose pull source lies beyond the inflow plane x = 0 carry the VBB code of side 0, nothing else does
    for i in range(1, Q):
        crossing = ix - cx[i] < 0
        assert (nb[crossing, i - 1] == O.LINK_VBB0 - 0).all() and (nb[~crossing, i - 1] != O.LINK_VBB0 - 0).all()
    gained_uniform = []
    for step in range(5):
        f = g.populations(0, 0)
        rho_cell = f.sum(axis=1)
        expect = sum(2.0 * w[i] * (cx[i] * u_in) / cs2 * rho_cell[ix - cx[i] < 0].sum() for i in range(1, Q))
        assert g.step(1) == 0
        gain = g.populations(0, 0).sum() - f.sum()
        assert abs(gain - expect) < 1e-13, (step, gain, expect)
        gained_uniform.append(expect / (u_in * ny))
    # and that sum is rho u_in per unit height up to the inlet's density variation
    assert all(abs(x - 1.0) < 0.1 for x in gained_uniform)
    # uniform density: exactly rho u_in ny per step
    def flat(level, ix, iy):
        o = np.ones(len(ix))
        return 1.3 * o, 0 * o, 0 * o, cs2 * o
    case.fields = flat
    g = oracle_from_case(case)
    m0 = g.populations(0, 0).sum()
    assert g.step(1) == 0
    assert abs((g.populations(0, 0).sum() - m0) - 1.3 * u_in * ny) < 1e-13
