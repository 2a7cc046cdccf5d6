"""GPU parity of the three addressing modes of the sweep on grids small enough for the oracle
to follow for many steps: regular bricks forced on small levels (lbm_config.addressing = LBM_ADDR_BRICKS; by default
only levels of >= 2^18 cells use them, which the full-size tests cover), the default small-level mode (list, one cell per
thread), and the list-only kernel (LBM_ADDR_LIST; fp32: two cells per thread)."""
import numpy as np
import pytest

from helpers import gpu_from_case, max_pop_diff, oracle_from_case
from paper_2504_04465_b200 import workloads as W

pytestmark = pytest.mark.gpu

MODES = {"bricks": dict(addressing=2), "small": dict(addressing=0), "list_only": dict(addressing=1)}   # LBM_ADDR_*
TOL = {64: 1e-12, 32: 1e-5}


def _fields(nc, depth, cs2):
    n = nc << depth
    k = 2 * np.pi / n

    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        return (1.0 + 0.03 * np.sin(k * x) * np.cos(k * y), 0.04 * np.sin(k * y), -0.03 * np.cos(k * x + k * y), np.full(len(x), cs2))
    return fields


def _cases():
    return {
        "tgv40_bgk": (lambda: W.tgv(40), 20),                                   # ragged: 25 whole tiles of 8x8 in a 40^2 periodic box
        "tgv64_rr": (lambda: W.tgv(64, collision=W.RR), 20),
        "cavity": (lambda: W.cavity(), 10),                                     # walls, moving lid, 2 levels
        "cylinder_small": (lambda: W.cylinder(D=40, depth=3, radii=(3, 5, 8)), 3),
        "cylinder_sponge": (lambda: W.cylinder(D=40, depth=3, radii=(3, 5, 8), sponge_d=(24, 30, 0.1)), 3),   # Eq. 10-11
        "patch_q13": (lambda: W.patch(nc=64, lo=16, hi=48, lattice=13, collision=W.RR, tau0=0.7, fields=_fields(64, 1, 0.5)), 4),
        "patch_q21": (lambda: W.patch(nc=64, lo=16, hi=48, lattice=21, collision=W.BGK, tau0=0.7, fields=_fields(64, 1, 2.0 / 3.0)), 4),
        "riemann_q37_ddf_sensor": (lambda: W.riemann(n=64), 3),                 # Neumann layers; fp64 only (as in test_gpu_parity)
        "riemann_q37_periodic": (lambda: W.riemann(n=48, periodic=True), 3),
    }


@pytest.mark.parametrize("mode", sorted(MODES))
@pytest.mark.parametrize("name", sorted(_cases()))
def test_addressing_modes_match_the_oracle(name, mode):
    make, ncoarse = _cases()[name]
    case = make()
    o = oracle_from_case(case)
    assert o.step(ncoarse) == 0
    for prec in ((64,) if case.ddf else (64, 32)):
        g = gpu_from_case(case, prec, **MODES[mode])
        if mode == "bricks":
            assert sum(int(g.info.n_bricks[l]) for l in range(g.depth + 1)) > 0
            assert "bricks" in g.kernel_name()
        if mode == "list_only":
            assert "bricks" not in g.kernel_name()
        g.step(ncoarse)
        assert g.sync() == 0
        d = max_pop_diff(g, o, (0, 1) if case.ddf else (0,))
        assert d <= TOL[prec], (name, mode, prec, d)
        g.close()
