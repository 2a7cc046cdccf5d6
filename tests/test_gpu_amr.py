"""GPU parity of lbm_transfer (mesh adaptation, Sec. 8.1 of the paper P:696-698; transfer_kernel of csrc/lbm_api.cu: look-up and transfer on the device)
against the oracle's orc_transfer on the same pairs of trees: a refined patch that moves and deepens (copy, explosion,
coalescence over one and two levels, ghost bands on both sides), the graded cylinder mesh with other radii (solid cells:
N_f < 4, inflow / Neumann boundary cells), the NACA mesh with numerical equilibria (g and the multipliers lambda move too,
Dirichlet and Neumann cells), both precisions; then both sides keep stepping on the new tree and are compared again."""
import numpy as np
import pytest

from helpers import gpu_from_case, max_pop_diff, oracle_from_case
from paper_2504_04465_b200 import lbm, workloads as W

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5}


def _fields(n):
    k = 2 * np.pi / n

    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        return (1.0 + 0.05 * np.sin(k * x) * np.cos(k * y), 0.06 * np.sin(k * y), -0.04 * np.cos(k * x), np.full(len(x), 1.0 / 3.0))
    return fields


def _patch(lo, hi, d):
    return W.patch(nc=128 >> d, lo=lo, hi=hi, depth=d, lattice=9, collision=W.RR, tau0=0.7, fields=_fields(128))


PAIRS = {
    "patch_moves": (lambda: _patch(16, 48, 1), lambda: _patch(8, 40, 1), (64, 32)),
    "patch_deepens": (lambda: _patch(16, 48, 1), lambda: _patch(4, 28, 2), (64, 32)),
    "patch_coarsens_two_levels": (lambda: _patch(4, 28, 2), lambda: W.Case("u", W.Mesh(2, 32, 32, [None] * 3, [None] * 3), lattice=9,
                                                                        collision=W.RR, tau0=0.7, fields=_fields(128)), (64,)),
    "cylinder_radii": (lambda: W.cylinder(D=40, depth=3, radii=(3, 5, 8)), lambda: W.cylinder(D=40, depth=3, radii=(2, 6, 9)), (64, 32)),
    "naca_numeq_radii": (lambda: W.naca(chord=64, depth=3, radii=(1, 2.5, 5), aoa_deg=4.0),
                         lambda: W.naca(chord=64, depth=3, radii=(1.5, 3, 4.5), aoa_deg=4.0), (64,)),
}


@pytest.mark.parametrize("name", sorted(PAIRS))
def test_transfer_matches_the_oracle_and_the_run_continues(name):
    mk_old, mk_new, precisions = PAIRS[name]
    old, new = mk_old(), mk_new()
    which = (0, 1, 2) if old.collision == W.NUMEQ else (0, 1) if old.ddf else (0,)
    oo = oracle_from_case(old)
    assert oo.step(2) == 0
    on = oracle_from_case(new, init=False)
    assert on.transfer_from(oo) == 0
    for prec in precisions:
        go = gpu_from_case(old, prec)
        go.step(2)
        assert go.sync() == 0
        gn = gpu_from_case(new, prec, init=False)
        gn.transfer_from(go)
        assert gn.sync() == 0
        d = max_pop_diff(gn, on, which)
        assert d <= TOL[prec], (name, prec, "transfer", d)
        go.close()
    assert on.step(2) == 0
    gn.step(2)                                   # the last precision's grid keeps running on the new tree
    assert gn.sync() == 0
    d = max_pop_diff(gn, on, which[:2])
    assert d <= TOL[precisions[-1]] * 2, (name, "after two more coarse steps", d)
    gn.close()


def test_transfer_onto_the_same_tree_is_bit_exact_and_errors_are_reported():
    case = W.cylinder(D=40, depth=3, radii=(3, 5, 8))
    a = gpu_from_case(case, 64)
    a.step(1)
    b = gpu_from_case(case, 64, init=False)
    b.transfer_from(a)
    for l in range(a.depth + 1):
        assert np.array_equal(a.populations(l), b.populations(l))
    a.step_fine(1)                               # inside a coarse step: not a re-mesh point
    with pytest.raises(lbm.LbmError) as e:
        b.transfer_from(a)
    assert e.value.code == lbm.ESTATE
    free = W.cylinder(D=40, depth=3, radii=(3, 5, 8))
    free.mesh.solid[0] = None
    c = gpu_from_case(free, 64, init=False)
    a.step_fine((1 << a.depth) - 1)
    with pytest.raises(lbm.LbmError) as e:
        c.transfer_from(a)
    assert e.value.code == lbm.EMESH
    d = gpu_from_case(W.cylinder(D=40, depth=3, radii=(3, 5, 8), lattice=13), 64, init=False)
    with pytest.raises(lbm.LbmError) as e:
        d.transfer_from(a)
    assert e.value.code == lbm.EINVAL
    for g in (a, b, c, d):
        g.close()


SENSOR_CASES = {
    "stripe_q9_rr": (lambda: W.stripe(nc=32, lo=8, hi=24, lattice=9, collision=W.RR, tau0=0.6, fields=_fields(64)), {}),
    "cavity_matrix": (lambda: W.cavity_uniform(64), dict(addressing=lbm.ADDR_MATRIX)),
    "riemann_q37_ddf": (lambda: W.riemann(n=48), {}),
    "naca_numeq": (lambda: W.naca(chord=64, depth=3, radii=(1, 2.5, 5), mach=1.5), {}),
}


@pytest.mark.parametrize("name", sorted(SENSOR_CASES))
def test_sensor_field_matches_the_oracle(name):
    """lbm_get_sensor (the refinement criterion of P:717, Eq. 52 on the stored state) against orc_get_sensor."""
    mk, opts = SENSOR_CASES[name]
    case = mk()
    o = oracle_from_case(case)
    assert o.step(3) == 0
    eo = o.sensor()
    for prec in ((64, 32) if name in ("stripe_q9_rr", "cavity_matrix") else (64,)):
        g = gpu_from_case(case, prec, **opts)
        g.step(3)
        assert g.sync() == 0
        eg = g.sensor()
        assert eo.max() > 1e-6                                          # the case has something to sense
        assert np.abs(eg - eo).max() <= (1e-10 if prec == 64 else 2e-5), (name, prec, np.abs(eg - eo).max())
        g.close()


def test_sensor_driven_adaptation_follows_a_convected_vortex():
    """The adaptive cycle of Sec. 8 of the paper end to end (its Fig. 26 case in miniature): a vortex convected through a
    periodic box on a two-level tree whose fine patch is rebuilt every four coarse steps from the kinetic sensor computed on
    the device (cells above 30 % of its maximum, dilated by four coarse cells), the state moved by lbm_transfer.  The oracle
    runs the same cycle on the same flags (they are inputs, passed in); both are compared after every re-mesh and at the
    end, mass is conserved to rounding, and the patch travels with the vortex."""
    nc, u0 = 64, 0.08
    L = 2 * nc

    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        dx, dy = x - 0.3 * L, y - 0.5 * L
        r2 = (dx * dx + dy * dy) / (0.06 * L) ** 2
        a = 0.06 * np.exp(0.5 * (1.0 - r2))
        return 1.0 - 0.5 * a * a * 3.0, u0 - a * dy / (0.06 * L), a * dx / (0.06 * L), np.full(len(x), 1.0 / 3.0)

    def case_of(mask):
        mesh = W.build_mesh(1, nc, nc, lambda level, ix, iy: mask[iy, ix])
        return W.Case("amr", mesh, lattice=9, collision=W.RR, tau0=0.52, fields=fields)

    def flags(g):
        e = g.sensor()
        E = np.zeros((nc, nc))
        for l in (0, 1):
            ix, iy, ty, _ = g.cells(l)
            np.maximum.at(E, (iy >> (1 - l), ix >> (1 - l)), e[g.off[l]:g.off[l + 1]])
        m = E > 0.3 * E.max()
        out = np.zeros_like(m)
        for sx in range(-4, 5):
            for sy in range(-4, 5):
                out |= np.roll(np.roll(m, sx, axis=1), sy, axis=0)
        return out

    yy, xx = np.mgrid[0:nc, 0:nc]
    mask = (xx - 0.3 * nc) ** 2 + (yy - 0.5 * nc) ** 2 < 10 ** 2
    case = case_of(mask)
    g, o = gpu_from_case(case, 64), oracle_from_case(case)
    mass0 = sum(4.0 ** l * g.populations(l)[np.isin(g.cells(l)[2], (lbm.FLUID, lbm.COARSE_GHOST))].sum() for l in (0, 1))
    centroids = []
    for cycle in range(5):
        g.step(4)
        assert g.sync() == 0 and o.step(4) == 0
        mask = flags(g)
        centroids.append(float((xx[mask] * 1.0).mean()))
        case = case_of(mask)
        g2, o2 = gpu_from_case(case, 64, init=False), oracle_from_case(case, init=False)
        g2.transfer_from(g)
        assert o2.transfer_from(o) == 0
        g.close()
        g, o = g2, o2
        assert max_pop_diff(g, o) <= 1e-12, cycle
    g.step(4)
    assert g.sync() == 0 and o.step(4) == 0
    assert max_pop_diff(g, o) <= 1e-12
    mass1 = sum(4.0 ** l * g.populations(l)[np.isin(g.cells(l)[2], (lbm.FLUID, lbm.COARSE_GHOST))].sum() for l in (0, 1))
    assert abs(mass1 - mass0) <= 1e-6 * mass0          # Rohde coupling + re-meshing: the corner leak of S8b only
    shift = centroids[-1] - centroids[0]                 # 16 coarse steps x 2 fine steps x u0 = 2.56 fine = 1.28 coarse cells downstream
    assert 0.8 < shift < 1.8, centroids
    g.close()
