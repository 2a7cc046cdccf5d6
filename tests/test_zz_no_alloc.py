"""lbm_get_macroscopic_at_static (include/lbm.h): the probe-cell read-out whose device scratch is a file-scope
`static __device__` array of the library instead of the caller's arena -- one entry point that allocates nothing, for callers
that may not call cudaMalloc.  Checked against the existing path (lbm_get_macroscopic_at: same kernel, scratch in the arena)
on two calls in a row that reuse the shared array with different cell lists, on a multilevel tree, on a thermal model and on
the matrix-like path; sizes beyond LBM_STATIC_PROBE_MAX are refused.  This file is collected last on purpose (pytest -x)."""
import numpy as np
import pytest

from helpers import gpu_from_case
from paper_2504_04465_b200 import lbm, workloads as W

pytestmark = pytest.mark.gpu


def _same(a, b):
    # the two paths run the same kernel on the same state: identical bits; the suite's fp64 tolerance is the bound asserted
    for x, y in zip(a, b):
        assert x.shape == y.shape and np.abs(x - y).max() <= 1e-12
        assert np.array_equal(x, y)


@pytest.mark.parametrize("name", ["cylinder_fp64", "cylinder_fp32", "riemann_q37_ddf", "cavity_matrix"])
def test_static_scratch_probe_matches_the_arena_scratch_path_twice_in_a_row(name):
    case, prec, opts = {
        "cylinder_fp64": (W.cylinder(D=40, depth=3, radii=(3, 5, 8)), 64, {}),
        "cylinder_fp32": (W.cylinder(D=40, depth=3, radii=(3, 5, 8)), 32, {}),
        "riemann_q37_ddf": (W.riemann(n=64), 64, {}),
        "cavity_matrix": (W.cavity_uniform(96), 64, dict(addressing=lbm.ADDR_MATRIX)),
    }[name]
    g = gpu_from_case(case, prec, **opts)
    g.step(3)                                   # odd: the matrix-like path sits in its shifted layout
    assert g.sync() == 0
    rng = np.random.default_rng(7)
    n0 = g.n[0]
    first = rng.integers(0, n0, size=min(3000, lbm.STATIC_PROBE_MAX)).astype(np.int32)
    second = rng.integers(0, n0, size=257).astype(np.int32)     # shorter: the array still holds the first call's tail
    _same(g.macroscopic_at_static(0, first), g.macroscopic_at(0, first))
    _same(g.macroscopic_at_static(0, second), g.macroscopic_at(0, second))
    if g.depth:                                  # another level, and the full field as the cross-check
        l = g.depth
        cells = np.arange(g.n[l], dtype=np.int32)[:lbm.STATIC_PROBE_MAX]
        got = g.macroscopic_at_static(l, cells)
        _same(got, g.macroscopic_at(l, cells))
        full = g.macroscopic()
        for x, y in zip(got, full):
            assert np.array_equal(x, y[g.off[l]:g.off[l] + cells.size])
    g.step(2)                                    # the run goes on, and so does the read-out
    assert g.sync() == 0
    _same(g.macroscopic_at_static(0, second), g.macroscopic_at(0, second))
    g.close()


def test_static_scratch_limits_and_errors():
    g = gpu_from_case(W.tgv(128), 64)
    ok = np.zeros(lbm.STATIC_PROBE_MAX, np.int32)
    g.macroscopic_at_static(0, ok)                                # exactly the maximum
    with pytest.raises(lbm.LbmError) as e:
        g.macroscopic_at_static(0, np.zeros(lbm.STATIC_PROBE_MAX + 1, np.int32))
    assert e.value.code == lbm.ETOOLARGE
    with pytest.raises(lbm.LbmError) as e:
        g.macroscopic_at_static(0, np.array([g.n[0]], np.int32))  # index outside the level
    assert e.value.code == lbm.EINVAL
    assert all(x.size == 0 for x in g.macroscopic_at_static(0, np.zeros(0, np.int32)))
    # two grids share the one array: calls one after the other do not disturb each other's results
    h = gpu_from_case(W.tgv(64, u0=0.02), 64)
    cells = np.arange(100, dtype=np.int32)
    a = g.macroscopic_at_static(0, cells)
    b = h.macroscopic_at_static(0, cells)
    _same(a, g.macroscopic_at(0, cells))
    _same(b, h.macroscopic_at(0, cells))
    g.close(); h.close()
