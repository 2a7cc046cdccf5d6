"""Every kernel set the library ships (csrc/sweep_q*.cu, enumerated through lbm_supported_model) has a parity case: a
two-level periodic stripe (two straight interfaces: coalescence, explosion, fine ghosts, asynchronous schedule) with a
smooth non-uniform field, two coarse steps, compared with the oracle element by element (f, and g where the model has
one) at north_star's tolerances; polynomial models in both addressing modes (list and regular bricks), the wide models
(second distribution and / or numerical equilibria) also through the software-pipelined sweep with a grid of three CTAs, so
that every thread walks over several cells."""
import numpy as np
import pytest

from helpers import gpu_from_case, max_pop_diff, oracle_from_case
from paper_2504_04465_b200 import lbm, workloads as W

TOL = {64: 1e-12, 32: 1e-5}
T0_NUMEQ = {13: 0.35, 21: 0.65, 37: 0.4}       # reference temperatures of the paper's runs


def _sets():
    """The shipped sets, written out (a CPU test below checks this list against the library's own enumeration)."""
    out = []
    for Q in (9, 13, 21):
        out += [(Q, 64, W.BGK, 0, 0), (Q, 64, W.RR, 0, 0), (Q, 32, W.BGK, 0, 0), (Q, 32, W.RR, 0, 0)]
    for Q in (13, 21):
        out += [(Q, 64, W.BGK, 1, 0), (Q, 64, W.BGK, 1, 1), (Q, 64, W.NUMEQ, 0, 0), (Q, 64, W.NUMEQ, 1, 0), (Q, 64, W.NUMEQ, 1, 1),
                (Q, 32, W.NUMEQ, 1, 0), (Q, 32, W.NUMEQ, 1, 1)]
    out += [(37, 64, W.BGK, 0, 0), (37, 64, W.RR, 0, 0), (37, 32, W.BGK, 0, 0), (37, 32, W.RR, 0, 0), (37, 64, W.BGK, 1, 0), (37, 64, W.BGK, 1, 1), (37, 32, W.BGK, 1, 1),
            (37, 64, W.NUMEQ, 1, 0), (37, 64, W.NUMEQ, 1, 1), (37, 32, W.NUMEQ, 1, 1)]
    return out


def test_the_list_of_kernel_sets_is_the_librarys():
    assert sorted(_sets()) == sorted(lbm.supported_models())


def _case(Q, coll, ddf, sensor):
    nc = 48
    thermal = bool(ddf) or coll == W.NUMEQ
    T0 = T0_NUMEQ[Q] if coll == W.NUMEQ else W.CS2[Q]
    L = nc << 1
    k = 2 * np.pi / L

    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        rho = 1.0 + 0.05 * np.sin(k * x) * np.cos(2 * k * y)
        ux = 0.08 * np.sin(k * y + 0.3) + 0.02
        uy = -0.05 * np.cos(k * x) + 0.01
        T = T0 * (1.0 + (0.06 * np.cos(k * x + k * y) if thermal else 0.0))
        return rho, ux, uy, T
    return W.stripe(nc=nc, lo=12, hi=36, lattice=Q, collision=coll, ddf=ddf, sensor=sensor, tau0=0.62,
                    T0=(T0 if coll == W.NUMEQ else 0.0), sensor_A=1.35, fields=fields)


@pytest.mark.gpu
@pytest.mark.parametrize("Q,precision,coll,ddf,sensor", _sets())
def test_kernel_set_matches_the_oracle(Q, precision, coll, ddf, sensor):
    case = _case(Q, coll, ddf, sensor)
    o = oracle_from_case(case)
    which = (0, 1) if ddf else (0,)
    assert o.step(2) == 0
    for addressing in ((lbm.ADDR_LIST,) if coll == W.NUMEQ else (lbm.ADDR_LIST, lbm.ADDR_BRICKS)):
        g = gpu_from_case(case, precision, addressing=addressing)
        assert ("bricks" in g.kernel_name()) == (addressing == lbm.ADDR_BRICKS)
        g.step(2)
        assert g.sync() == 0
        d = max_pop_diff(g, o, which)
        assert d <= TOL[precision], (g.kernel_name(), d)
        g.close()
    if ddf or coll == W.NUMEQ:
        g = gpu_from_case(case, precision, pipeline=lbm.PIPE_ALWAYS, pipe_max_ctas=3)
        assert "sweep_pipe_kernel" in g.kernel_name()
        g.step(2)
        assert g.sync() == 0
        d = max_pop_diff(g, o, which)
        assert d <= TOL[precision], (g.kernel_name(), d)
        g.close()
