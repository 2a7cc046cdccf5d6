"""Physics pin of the fully compressible path of the ORACLE (numerical equilibrium Eq. 39-49, second distribution
Eq. 50-51 with gamma = 7/5, kinetic sensor Eq. 52-53, inviscid tau = 1/2, Neumann ends): the Sod shock tube of
Sec. 6.1 (Eq. 12) against the EXACT solution of the 1-D Riemann problem of the Euler equations (rarefaction,
contact, shock; the textbook two-wave pressure equation solved by bisection below).  The paper reports that "all
density profiles match very well the analytical solution" for D2Q13, D2Q21 and D2Q37; a wrong energy
coupling, a wrong gamma, a wrong moment constraint or a wrong streaming direction moves the three waves and fails
this test by an order of magnitude."""
import numpy as np
import pytest

from helpers import oracle_from_case
from paper_2504_04465_b200 import workloads as W

GAMMA = 1.4


def exact_riemann_density(xi, left, right, gamma=GAMMA):
    """rho(x/t) of the exact Riemann solution for a left rarefaction / right shock pattern; states are (rho, u, p)."""
    (rl, ul, pl), (rr, ur, pr) = left, right
    cl, cr = np.sqrt(gamma * pl / rl), np.sqrt(gamma * pr / rr)
    g1, g2, g3 = (gamma - 1) / (2 * gamma), (gamma + 1) / (2 * gamma), (gamma - 1) / (gamma + 1)

    def f(p, r, pk, c):      # velocity jump across the wave on side K as a function of the star pressure
        if p > pk:
            return (p - pk) * np.sqrt(2 / ((gamma + 1) * r) / (p + g3 * pk))
        return 2 * c / (gamma - 1) * ((p / pk) ** g1 - 1)

    lo, hi = 1e-12, 10 * max(pl, pr)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if f(mid, rl, pl, cl) + f(mid, rr, pr, cr) + ur - ul > 0:
            hi = mid
        else:
            lo = mid
    ps = 0.5 * (lo + hi)
    us = 0.5 * (ul + ur) + 0.5 * (f(ps, rr, pr, cr) - f(ps, rl, pl, cl))
    assert pr < ps < pl
    rsl = rl * (ps / pl) ** (1 / gamma)                      # behind the rarefaction (isentropic)
    csl = cl * (ps / pl) ** g1
    rsr = rr * ((ps / pr + g3) / (g3 * ps / pr + 1))         # behind the shock (Rankine-Hugoniot)
    s_shock = ur + cr * np.sqrt(g2 * ps / pr + g1)
    fan = rl * (2 / (gamma + 1) + g3 / cl * (ul - xi)) ** (2 / (gamma - 1))
    return np.where(xi < ul - cl, rl, np.where(xi < us - csl, fan, np.where(xi < us, rsl, np.where(xi < s_shock, rsr, rr)))), ps


def sod_l1_error(lattice, N):
    case = W.sod(L=N, lattice=lattice, mesh="unif", periodic=False, ny=8)
    o = oracle_from_case(case)
    T0 = W.SOD_T0[lattice]
    nsteps = int(round(0.2 * N / np.sqrt(GAMMA * T0)))       # t = 0.2 t_c, t_c = L / sqrt(gamma T0)
    assert o.step(nsteps) == 0
    rho = o.macroscopic()[0]
    ix, iy, ty, aux = o.cells(0)
    m = (iy == 3) & (ix >= 0) & (ix < N)
    order = np.argsort(ix[m])
    x = ix[m][order] + 0.5
    (rl, _, Tl), (rr, _, Tr) = case.meta["left"], case.meta["right"]
    exact, ps = exact_riemann_density((x - N / 2) / nsteps, (rl, 0.0, rl * Tl), (rr, 0.0, rr * Tr))
    assert abs(ps / (rr * Tr) - 3.0313) < 1e-3               # star pressure of the (10, 8) / (1, 1) tube
    # the tube is uniform in y: every row carries the same profile
    assert np.abs(rho[(iy == 5) & (ix >= 0) & (ix < N)][np.argsort(ix[(iy == 5) & (ix >= 0) & (ix < N)])] - rho[m][order]).max() < 1e-12
    return float(np.abs(rho[m][order] - exact).sum() / np.abs(exact).sum())


@pytest.mark.parametrize("lattice", [13, 21, 37])
def test_sod_shock_tube_matches_exact_riemann_solution(lattice):
    e128, e256 = sod_l1_error(lattice, 128), sod_l1_error(lattice, 256)
    assert e128 < 0.025 and e256 < 0.0125, (e128, e256)       # measured 0.013-0.019 and 0.008-0.010
    assert e256 < 0.65 * e128                                  # first-order convergence at the discontinuities
