"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same Case generators, same
precision switch, same graphs).  Where the oracle finishes in about a minute the comparison is element by element
over every stored cell of every level (uniform 4096^2, cylinder = configs[2] for one coarse step, riemann =
configs[3] for one step); for configs[4] (18 M cells of Newton solves: tens of minutes of oracle per coarse step)
it is on SAMPLED cells, each recomputed one by one by the oracle's cell routines from the CUDA path's own pre-step
state gathered through the bit-exact host neighbour list.  Tolerances: north_star (|df| <= 1e-12 fp64, 1e-5 fp32)."""
import numpy as np
import pytest

from helpers import gpu_from_case, max_pop_diff, oracle_from_case
from oracle import oracle as O
from paper_2504_04465_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5}


def _both_precisions(case, ncoarse, which):
    o = oracle_from_case(case)
    assert o.step(ncoarse) == 0
    out = {}
    for prec in (64, 32):
        g = gpu_from_case(case, prec)
        g.step(ncoarse)
        assert g.sync() == 0
        out[prec] = max_pop_diff(g, o, which)
        g.close()
    return out


def test_uniform_4096_one_step_all_cells():
    """bench.py --workload uniform: D2Q9-BGK, 16.8 M cells, tree-stored periodic box (configs[0] scaled)."""
    d = _both_precisions(W.tgv(4096), 1, (0,))
    assert d[64] <= TOL[64], d
    assert d[32] <= TOL[32], d


def test_uniform_4096_matrix_path_two_steps_all_cells():
    """bench.py --workload uniform --addressing matrix (the Eq. 14 point): Cartesian index + AA pattern, one even and one
    odd step, every cell, both precisions."""
    from paper_2504_04465_b200 import lbm
    case = W.tgv(4096)
    o = oracle_from_case(case)
    assert o.step(2) == 0
    for prec in (64, 32):
        g = gpu_from_case(case, prec, addressing=lbm.ADDR_MATRIX)
        g.step(2)
        assert g.sync() == 0
        d = max_pop_diff(g, o, (0,))
        assert d <= TOL[prec], (prec, d)
        g.close()


def test_cylinder_config3_one_coarse_step_all_cells():
    """bench.py default workload: configs[2], 6 levels, 9.8 M cells, 32 fine steps = 222 M cell updates: every
    interface coalesces and explodes 16..1 times, inflow / Neumann / bounce-back links included."""
    d = _both_precisions(W.cylinder(), 1, (0,))
    assert d[64] <= TOL[64], d
    assert d[32] <= TOL[32], d


def test_riemann_config4_one_step_all_cells():
    """bench.py --workload riemann: configs[3], D2Q37 polynomial + g + sensor on 2048^2 (+ Neumann layers)."""
    case = W.riemann(n=2048)
    o = oracle_from_case(case)
    assert o.step(1) == 0
    g = gpu_from_case(case, 64)
    g.step(1)
    assert g.sync() == 0
    d = max_pop_diff(g, o, (0, 1))
    assert d <= TOL[64], d


def _sample_cells(rng, ty, nbr, n_sample):
    """Fluid cells whose links are all cells or walls; half of the sample is taken among cells next to a wall."""
    ok = (ty == O.FLUID) & np.all((nbr >= 0) | (nbr == O.LINK_WALL), axis=1)
    wall = ok & np.any(nbr == O.LINK_WALL, axis=1)
    a = np.flatnonzero(ok)
    b = np.flatnonzero(wall)
    pick = [rng.choice(a, size=min(n_sample, a.size), replace=False)]
    if b.size:
        pick.append(rng.choice(b, size=min(n_sample, b.size), replace=False))
    return np.unique(np.concatenate(pick))


def test_naca_config5_sampled_cells_one_fine_step():
    """bench.py --workload naca: configs[4], D2Q21 numerical equilibrium + g + sensor, 7 levels, 18.3 M cells.
    (1) initialisation: the stored f, g of sampled cells against the oracle's Newton solve from the same start;
    (2) one fine step (level 0 updates): sampled cells recomputed by the oracle's collide routine from the CUDA
    path's pre-step populations and multipliers gathered through the host neighbour list (pull, Eq. 31; wall link =
    own opposite population)."""
    case = W.naca(chord=1024)
    g = gpu_from_case(case, 64)
    kw = case.model_kwargs()
    cfg = O.make_config(**kw)
    Q = 21
    cx, cy, w, opp, cs2, reach = O.lattice(Q)
    ix, iy, ty, aux = g.cells(0)
    nbr = g.nbr(0)
    rng = np.random.default_rng(20250404)
    cells = _sample_cells(rng, ty, nbr, 1500)
    assert cells.size >= 1500
    f0, g0, l0 = g.populations(0, 0), g.populations(0, 1), g.populations(0, 2)

    # (1) initial state of the sampled cells
    rho, ux, uy, T = W.eval_fields(case, [g.cells(l)[:2] for l in range(g.depth + 1)])
    fac = 2.0 / (kw["gamma"] - 1.0) - 2.0
    d_init = 0.0
    for c in cells[:300]:
        r, u, v, t = rho[c], ux[c], uy[c], T[c]          # level 0 comes first in the flat arrays
        start = [(u * u + v * v) / (2 * t) + np.log(2 * np.pi * t) - 1, -u / t, -v / t, 1 / (2 * t), 0.0, 1 / (2 * t), 0.0, 0.0]
        fe, lam, it = O.feq_numerical(Q, r, u, v, t, lam=start, tol=kw["newton_tol"], max_iter=kw["newton_max_iter"])
        assert it >= 0
        d_init = max(d_init, np.abs(f0[c] - fe).max(), np.abs(g0[c] - fac * t * fe).max())
    assert d_init <= TOL[64], d_init

    # (2) one fine step
    g.step_fine(1)
    assert g.sync() == 0
    f1, g1 = g.populations(0, 0), g.populations(0, 1)
    tau0 = g.info.tau[0]
    d_step = 0.0
    for c in cells:
        fin = np.empty(Q)
        gin = np.empty(Q)
        fin[0], gin[0] = f0[c, 0], g0[c, 0]
        for i in range(1, Q):
            s = nbr[c, i - 1]
            if s >= 0:
                fin[i], gin[i] = f0[s, i], g0[s, i]
            else:
                fin[i], gin[i] = f0[c, opp[i]], g0[c, opp[i]]
        fo, go, lam, it = O.collide_cell(cfg, tau0, fin, gin, l0[c])
        assert it >= 0
        d_step = max(d_step, np.abs(f1[c] - fo).max(), np.abs(g1[c] - go).max())
    assert d_step <= TOL[64], d_step
    # the remaining fine steps of the coarse step run through the same ABI call; then graphs may resume
    g.step_fine((1 << g.depth) - 1)
    g.step(1)
    assert g.sync() == 0
    g.close()


def test_naca_config5_all_levels_all_cells_one_fine_step():
    """configs[4] at full size, EVERY stored cell of all 7 levels (18.3 M: fluid, coarse and fine ghosts of six interfaces,
    Dirichlet and Neumann cells, walls of the airfoil): the CUDA path runs 63 fine steps of the schedule, its complete
    state (f, g, lambda of every level) is handed to the oracle, and both take fine step 64 -- the one in which all levels
    update, level 0 first: every coalescence (f, g and the multiplier warm start of Eq. 6), collision with the Newton
    solve, explosion (Eq. 5, 7) and boundary cell of the mesh, in the launch configuration bench.py times."""
    case = W.naca(chord=1024)
    g = gpu_from_case(case, 64)
    nf = 1 << g.depth
    g.step_fine(nf - 1)
    assert g.sync() == 0
    o = oracle_from_case(case, init=False)
    assert o.n == g.n
    for l in range(g.depth + 1):
        for w in (0, 1, 2):
            o.set_populations(l, w, g.populations(l, w))
    assert o.set_fine_step(nf - 1) == 0
    g.step_fine(1)
    assert g.sync() == 0
    assert o.step_fine(1) == 0
    worst = {}
    for l in range(g.depth + 1):
        ty = g.cells(l)[2]
        for w in (0, 1, 2):
            d = np.abs(g.populations(l, w) - o.populations(l, w)).max(axis=1)
            for t in np.unique(ty):
                worst[(w, int(t))] = max(worst.get((w, int(t)), 0.0), float(d[ty == t].max()))
    assert {t for (_, t) in worst} == {O.FLUID, O.FINE_GHOST, O.COARSE_GHOST, O.NEUMANN, O.DIRICHLET}
    assert max(v for (w, _), v in worst.items() if w < 2) <= TOL[64], worst
    assert max(v for (w, _), v in worst.items() if w == 2) <= 1e-9, worst
    g.step(1)                                   # the schedule is back at a coarse-step boundary: graphs resume
    assert g.sync() == 0
    g.close()
