"""GPU parity of lbm_transfer (mesh adaptation, Sec. 8.1 of the paper P:696-698; csrc/transfer.cpp + transfer_kernel)
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
