"""Pins of the oracle's mesh-adaptation transfer (oracle/amr.c; Sec. 8.1 of the paper: copy where the old tree
stores the cell, uniform explosion for refinement, conservative coalescence for coarsening).  None of them repeats its
code: they are what the paper and the arithmetic fix --
 A1  a transfer onto the same tree is the identity, bit for bit (every cell "finds a match");
 A2  a uniform state (any lattice, with g and lambda) survives any re-mesh: copies, explosions and means never leave the
     range of the old values (the old ghost cells differ from the leaves by the rounding of one collision, so the bound
     is that spread, a few ulp, not zero);
 A3  mass, momentum and energy summed over the leaves (weighted by cell area) are the same before and after, to rounding:
     explosion copies a density onto the same area, coalescence is the arithmetic mean ("conservative", Eq. 4-5);
 A4  refining a region and coarsening it again returns the original leaf values (mean of four copies), and a refined
     cell's children all carry the parent's state (Eq. 5: uniform explosion), the coarsened cell the mean of its four
     children computed here with numpy (Eq. 4);
 A5  a tree whose solids differ has cells without data: ORC_EMESH."""
import numpy as np
import pytest

from helpers import conserved_sums, oracle_from_case
from oracle import oracle as O
from paper_2504_04465_b200 import workloads as W


def _fields(n):
    k = 2 * np.pi / n

    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        return (1.0 + 0.05 * np.sin(k * x) * np.cos(k * y), 0.06 * np.sin(k * y), -0.04 * np.cos(k * x), np.full(len(x), 1.0 / 3.0))
    return fields


def _patch(lo, hi, depth=1, **kw):
    return W.patch(nc=32, lo=lo, hi=hi, depth=depth, fields=_fields(32 << depth), **kw)


def _state(o):
    return [np.concatenate([o.populations(l, w) for w in ((0, 1, 2) if o.cfg.collision == O.NUMEQ else (0, 1) if o.cfg.ddf else (0,))], axis=1)
            for l in range(o.depth + 1)]


def test_A1_same_tree_is_the_identity():
    a = oracle_from_case(_patch(8, 24))
    assert a.step(3) == 0
    b = oracle_from_case(_patch(8, 24), init=False)
    assert b.transfer_from(a) == 0
    for sa, sb in zip(_state(a), _state(b)):
        assert np.array_equal(sa, sb)
    assert a.step(2) == 0 and b.step(2) == 0          # and the run continues identically
    for sa, sb in zip(_state(a), _state(b)):
        assert np.array_equal(sa, sb)


@pytest.mark.parametrize("model", ["q9", "q21_numeq_ddf", "q37_poly_ddf"])
def test_A2_uniform_state_survives_any_remesh(model):
    kw = {"q9": dict(lattice=9, collision=W.RR),
          "q21_numeq_ddf": dict(lattice=21, collision=W.NUMEQ, ddf=1, sensor=1, T0=0.65),
          "q37_poly_ddf": dict(lattice=37, collision=W.BGK, ddf=1)}[model]
    T = 0.65 if model == "q21_numeq_ddf" else W.CS2[kw["lattice"]]

    def uniform(level, ix, iy):
        o = np.ones(len(ix))
        return 1.1 * o, 0.07 * o, -0.03 * o, T * o
    mk = lambda lo, hi, d: W.patch(nc=64 >> d, lo=lo, hi=hi, depth=d, fields=uniform, tau0=0.7, **kw)
    a = oracle_from_case(mk(8, 24, 1))
    old = np.concatenate([s for s in _state(a) if len(s)])
    lo_old, hi_old = old.min(axis=0), old.max(axis=0)
    assert (hi_old - lo_old).max() <= 1e-13      # D2Q37: the 15-digit weights of Table 4 leave collide(f_eq) - f_eq ~ 1e-14
    for lo, hi, d in ((4, 20, 1), (1, 15, 2), (0, 0, 0)):        # moved, deeper, no refinement at all (uniform finest grid)
        b = oracle_from_case(mk(lo, hi, d) if d else W.Case("u", W.uniform_mesh(64, 64), fields=uniform, tau0=0.7, **kw), init=False)
        assert b.transfer_from(a) == 0
        for s in _state(b):
            if len(s):
                assert np.all(s >= lo_old - 1e-17) and np.all(s <= hi_old + 1e-17)


@pytest.mark.parametrize("lattice", [9, 21])
def test_A3_mass_momentum_energy_are_conserved(lattice):
    kw = dict(lattice=lattice, collision=W.RR, tau0=0.7)
    a = oracle_from_case(W.patch(nc=32, lo=8, hi=24, depth=1, fields=_fields(64), **kw))
    assert a.step(2) == 0
    before = conserved_sums(a)
    for lo, hi, d in ((4, 20, 1), (12, 30, 1), (1, 15, 2)):
        b = oracle_from_case(W.patch(nc=64 >> d, lo=lo, hi=hi, depth=d, fields=_fields(64), **kw), init=False)
        assert b.transfer_from(a) == 0
        after = conserved_sums(b)
        assert np.abs(after - before).max() <= 2e-12 * np.abs(before).max(), (lo, hi, d, after - before)


def test_A4_explosion_copies_the_parent_coalescence_is_the_mean_of_the_children():
    coarse = oracle_from_case(W.Case("u", W.uniform_mesh(16, 16), lattice=9, collision=W.BGK, tau0=0.8, fields=_fields(16)))
    assert coarse.step(2) == 0
    # refine everything once: a uniform level-0 grid of 32 x 32 over the same box
    fine = oracle_from_case(W.Case("u", W.uniform_mesh(32, 32), lattice=9, collision=W.BGK, tau0=0.8, fields=_fields(32)), init=False)
    # the two trees must describe the same box: 16 cells of size 2 = depth-1 tree without split cells
    coarse1 = oracle_from_case(W.Case("u", W.Mesh(1, 16, 16, [None, None], [None, None]), lattice=9, collision=W.BGK, tau0=0.8, fields=_fields(32)))
    assert coarse1.step(2) == 0
    assert fine.transfer_from(coarse1) == 0
    Sc, Sf = coarse1.populations(1), fine.populations(0)
    cx, cy = coarse1.cells(1)[:2]
    fx, fy = fine.cells(0)[:2]
    parent = {(int(x), int(y)): k for k, (x, y) in enumerate(zip(cx, cy))}
    for k in range(0, len(fx), 7):
        assert np.array_equal(Sf[k], Sc[parent[(int(fx[k]) >> 1, int(fy[k]) >> 1)]])       # Eq. 5
    # and back: the mean of four copies is the original, bit for bit
    back = oracle_from_case(W.Case("u", W.Mesh(1, 16, 16, [None, None], [None, None]), lattice=9, collision=W.BGK, tau0=0.8, fields=_fields(32)), init=False)
    assert back.transfer_from(fine) == 0
    assert np.array_equal(back.populations(1), Sc)
    # coalescence of a non-uniform fine state = (1/4) sum of the four children (Eq. 4)
    assert fine.step(3) == 0
    Sf = fine.populations(0)
    child = {(int(x), int(y)): k for k, (x, y) in enumerate(zip(fx, fy))}
    assert back.transfer_from(fine) == 0
    Sb = back.populations(1)
    for k in range(0, len(cx), 5):
        x, y = int(cx[k]), int(cy[k])
        mean = (Sf[child[(2 * x, 2 * y)]] + Sf[child[(2 * x + 1, 2 * y)]] + Sf[child[(2 * x, 2 * y + 1)]] + Sf[child[(2 * x + 1, 2 * y + 1)]]) / 4
        assert np.array_equal(Sb[k], mean)


def test_A5_cells_without_old_data_are_an_error():
    a = oracle_from_case(W.cylinder(D=40, depth=3, radii=(3, 5, 8)))
    free = W.cylinder(D=40, depth=3, radii=(3, 5, 8))
    free.mesh.solid[0] = None                                   # the same tree without the cylinder
    b = oracle_from_case(free, init=False)
    assert b.transfer_from(a) == -3         # ORC_EMESH


# ----------------------------------------------------------------------------- the refinement criterion (Eq. 52)
def _d2q9_feq(rho, ux, uy):
    """Textbook D2Q9 second-order equilibrium in the canonical direction order, written out here (not the oracle's code);
    with the oracle's basis (Table 5: + xxy, xyy, xxyy terms) it is the product form: w_i rho prod_a (1 + 3 c_a u_a + ...)."""
    cx = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1]); cy = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])
    w = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)
    # product form of the extended-basis D2Q9 equilibrium: rho * psi_cx(ux) * psi_cy(uy), psi_0 = 2/3 (1 - 3u^2/2) ... with weights folded in
    px = np.where(cx == 0, (2 / 3) * (1 - 1.5 * ux * ux), (1 / 6) * (1 + 3 * cx * ux + 3 * ux * ux))
    py = np.where(cy == 0, (2 / 3) * (1 - 1.5 * uy * uy), (1 / 6) * (1 + 3 * cy * uy + 3 * uy * uy))
    return rho * px * py, cx, cy, w


def test_A6_sensor_is_the_relative_departure_from_equilibrium():
    case = W.Case("u", W.uniform_mesh(8, 8), lattice=9, collision=W.BGK, tau0=0.8,
                  fields=lambda l, ix, iy: (np.full(len(ix), 1.05), np.full(len(ix), 0.06), np.full(len(ix), -0.03), np.full(len(ix), 1 / 3)))
    o = oracle_from_case(case)
    assert np.abs(o.sensor()).max() <= 1e-13                       # equilibrium: eps = 0
    feq, cx, cy, w = _d2q9_feq(1.05, 0.06, -0.03)
    assert np.abs(o.populations(0)[0] - feq).max() <= 1e-15        # the closed form above is the state the oracle initialised
    delta = w * cx * cy                                            # a pure stress perturbation: no mass, no momentum
    assert abs(delta.sum()) < 1e-17 and abs((delta * cx).sum()) < 1e-17 and abs((delta * cy).sum()) < 1e-17
    for amp in (1e-3, 4e-3):
        o.set_populations(0, 0, np.tile(feq + amp * delta, (64, 1)))
        expect = amp * np.sum(np.abs(delta) / feq) / 9.0           # Eq. 52 by hand
        assert np.abs(o.sensor() - expect).max() <= 1e-12 * expect + 1e-16
    # Eq. 30: one BGK collision scales f - f^eq by (1 - 1/tau): the sensor of the post-collision state follows
    pre = feq + 2e-3 * delta
    post, _, _, _ = O.collide_cell(o.cfg, 0.8, pre)
    o.set_populations(0, 0, np.tile(post, (64, 1)))
    e_post = o.sensor()[0]
    o.set_populations(0, 0, np.tile(pre, (64, 1)))
    assert abs(e_post - abs(1 - 1 / 0.8) * o.sensor()[0]) <= 1e-14
