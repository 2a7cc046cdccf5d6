"""CPU checks of the boundary: the C-ABI library loads, exports every symbol include/lbm.h declares, and its
host grid builder (row a11 of SURVEY.md Sec. 8(a)) agrees BIT FOR BIT with the oracle's independent builder:
cells, types, neighbour lists, ghost lists, unknown masks and the level schedule (north_star: "neighbor lists
and level schedules must be bit-exact").  No compute call is made (there is no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import oracle as O
from paper_2504_04465_b200 import lbm, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "lbm.h")).read()
    declared = sorted(set(re.findall(r"\b(lbm_[a-z_0-9]+)\s*\(", hdr)))
    assert sorted(lbm.SYMBOLS) == declared
    L = lbm.lib()
    for s in declared:
        assert hasattr(L, s), s


def test_struct_layout_matches_header():
    # the ctypes mirror of lbm_config / lbm_grid_info has the size the C compiler gives the header's structs
    import subprocess
    import tempfile
    src = '#include <stdio.h>\n#include "lbm.h"\nint main(){printf("%zu %zu\\n", sizeof(lbm_config), sizeof(lbm_grid_info));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        p = os.path.join(d, "s.c")
        open(p, "w").write(src)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), p, "-o", os.path.join(d, "s")])
        a, b = map(int, subprocess.check_output([os.path.join(d, "s")]).split())
    assert a == C.sizeof(lbm.LbmConfig)
    assert b == C.sizeof(lbm.LbmGridInfo)


CASES = {
    "tgv64": lambda: W.tgv(64),
    "cavity": lambda: W.cavity(),
    "cavity_q13": lambda: W.cavity(scale=0.5, lattice=13),
    "cylinder_small": lambda: W.cylinder(D=40, depth=3, radii=(3, 5, 8)),
    "cylinder_sponge": lambda: W.cylinder(D=40, depth=3, radii=(3, 5, 8), sponge_d=(24, 30, 0.1)),
    "riemann_neumann": lambda: W.riemann(n=64),
    "riemann_periodic": lambda: W.riemann(n=48, periodic=True),
    "naca_small": lambda: W.naca(chord=64, depth=3, radii=(1, 2.5, 5), aoa_deg=4.0),
    "naca_supersonic": lambda: W.naca(chord=64, depth=2, radii=(1, 2.5), mach=1.5),
    "patch_q21": lambda: W.patch(lattice=21),
    "patch_depth2": lambda: W.patch(nc=48, lo=8, hi=40, depth=2),
    "stripe_q37": lambda: W.stripe(lattice=37),
    "walled_patch": lambda: W.patch(periodic=False),
}


@pytest.mark.parametrize("name", sorted(CASES))
def test_host_builder_bit_exact_against_oracle_builder(name):
    case = CASES[name]()
    g = lbm.Grid.from_case(case)
    o = O.OracleGrid(O.make_config(**case.model_kwargs()), case.mesh.split, case.mesh.solid)
    assert g.n == o.n
    for l in range(g.depth + 1):
        for a, b in zip(g.cells(l), o.cells(l)):
            assert np.array_equal(a, b)
        assert np.array_equal(g.nbr(l), o.nbr(l))
        assert g.tau(l) == o.tau(l)
        assert np.array_equal(g.sponge(l), o.sponge(l))          # Eq. 11 at the cell centres, bit for bit
        if l >= 1:
            for a, b in zip(g.ghosts(l), o.ghosts(l)):
                assert np.array_equal(a, b)
    for a, b in zip(g.schedule(), o.schedule()):
        assert np.array_equal(a, b)
    info = g.info
    assert info.updates_per_coarse_step == sum(g.n[l] << (g.depth - l) for l in range(g.depth + 1))
    g.close()


def _zpos(m):
    """(x, y) of Z-position m in an 8x8 tile, x in the even bits."""
    x = (m & 1) | ((m >> 1) & 2) | ((m >> 2) & 4)
    y = ((m >> 1) & 1) | ((m >> 2) & 2) | ((m >> 3) & 4)
    return x, y


@pytest.mark.parametrize("name", sorted(CASES))
def test_bricks_reproduce_the_oracle_neighbour_list(name):
    """Compressed addressing of the device path (lbm_get_bricks): every brick is an aligned 8x8 tile of FLUID cells
    with consecutive storage indices, and tile arithmetic reproduces the ORACLE builder's neighbour list for each of
    its cells and directions; the table itself is re-derived here from the lattice's velocities."""
    case = CASES[name]()
    g = lbm.Grid.from_case(case)
    o = O.OracleGrid(O.make_config(**case.model_kwargs()), case.mesh.split, case.mesh.solid)
    cx, cy, w, opp, cs2, reach = O.lattice(g.Q)
    mm = np.arange(64)
    for l in range(g.depth + 1):
        t9, tab = g.bricks(l)
        for i in range(1, g.Q):
            for m in range(64):
                x, y = _zpos(m)
                sx, sy = x - cx[i], y - cy[i]
                k = (0 if sx < 0 else 2 if sx > 7 else 1) + 3 * (0 if sy < 0 else 2 if sy > 7 else 1)
                z = [mz for mz in range(64) if _zpos(mz) == (sx & 7, sy & 7)][0]
                assert tab[i - 1, m] == (k << 6) | z
        if len(t9) == 0:
            continue
        ix, iy, ty, aux = o.cells(l)
        nbr = o.nbr(l)
        base = t9[:, 4]
        assert np.all(np.diff(base) >= 64)
        cells = base[:, None] + mm[None, :]
        assert np.all(ty[cells] == O.FLUID)
        assert np.all(o.sponge(l)[cells] == 0.0)                  # sponge cells go through the list path
        assert np.all(ix[base] % 8 == 0) and np.all(iy[base] % 8 == 0)
        x, y = _zpos(mm)
        assert np.array_equal(ix[cells], ix[base][:, None] + x[None, :])
        assert np.array_equal(iy[cells], iy[base][:, None] + y[None, :])
        for i in range(1, g.Q):
            k, z = tab[i - 1] >> 6, tab[i - 1] & 63
            assert np.array_equal(t9[:, k] + z[None, :], nbr[cells, i - 1])
    g.close()


@pytest.mark.parametrize("Q", [9, 13, 21, 37])
@pytest.mark.parametrize("cpt", [1, 2])
def test_brick_tile_arithmetic_of_the_device_path(Q, cpt):
    """The rule brick_update (csrc/sweep.cuh) uses instead of the table, restated here and checked against the table the
    host builder verified against the list: a thread owning `cpt` x-adjacent cells starting at (x0, y0) of its brick
    reaches at most one tile column beside the centre (west if x0 < 4, else east) and one tile row, so four tile bases
    suffice; a source is (crosses the column ? rowX[cy] : rowC[cy]) + colZ[d], d = (cell of the thread) - cx, with no
    column crossing for d = 0 (nor for d = 1 of a pair: x0 is even there)."""
    g = lbm.Grid.from_case(W.tgv(32, lattice=Q, collision=W.RR if Q != 37 else W.BGK))
    cx, cy, w, opp, cs2, reach = O.lattice(Q)
    assert reach <= 3                                           # W <= 3 < 4: what the one-column / one-row claim rests on
    _, tab = g.bricks(0)
    g.close()
    spread3 = lambda v: (v & 1) | ((v & 2) << 1) | ((v & 4) << 2)
    for m0 in range(0, 64, cpt):
        x0, y0 = _zpos(m0)
        assert cpt == 1 or x0 % 2 == 0
        kx, ky = (0 if x0 < 4 else 2), (0 if y0 < 4 else 6)
        # slots of brick_nb[9] (k = column + 3 * row, centre 4) the thread fetches: centre, side column, side row, corner
        bCC, bXC, bCY, bXY = 4, 3 + kx, 1 + ky, kx + ky
        for i in range(Q):
            sy = y0 - int(cy[i])
            zy = spread3(sy & 7) << 1
            py = cy[i] != 0 and not (0 <= sy <= 7)
            rowC, rowX = (bCY if py else bCC), (bXY if py else bXC)
            for j in range(cpt):
                d = j - int(cx[i])
                sx = x0 + d
                px = (d < 0 or d >= cpt) and not (0 <= sx <= 7)
                if not (d < 0 or d >= cpt):
                    assert 0 <= sx <= 7                         # the static no-crossing cases
                k, z = (rowX if px else rowC), zy + spread3(sx & 7)
                if i == 0:
                    assert (k, z) == (4, m0 + j)
                else:
                    e = int(tab[i - 1, m0 + j])
                    assert (k, z) == (e >> 6, e & 63), (Q, cpt, m0, j, i)


def test_brick_coverage_of_the_bench_shapes():
    """A periodic uniform box is all bricks; the graded cylinder mesh is mostly bricks on its fine levels."""
    g = lbm.Grid.from_case(W.tgv(64))
    assert int(g.info.n_bricks[0]) * 64 == g.n[0]
    g.close()
    g = lbm.Grid.from_case(W.cylinder(D=40))
    frac = [int(g.info.n_bricks[l]) * 64 / g.n[l] for l in range(g.depth + 1)]
    assert frac[0] > 0.8, frac
    g.close()


def test_invalid_arguments_are_rejected():
    with pytest.raises(lbm.LbmError) as e:
        lbm.Grid(lbm.make_config(lattice=10, nx_coarse=8, ny_coarse=8))
    assert e.value.code == lbm.EINVAL
    with pytest.raises(lbm.LbmError) as e:
        lbm.Grid(lbm.make_config(lattice=9, collision=lbm.RR, ddf=1, nx_coarse=8, ny_coarse=8))
    assert e.value.code == lbm.EINVAL
    with pytest.raises(lbm.LbmError) as e:
        lbm.Grid(lbm.make_config(lattice=9, tau0=0.4, nx_coarse=8, ny_coarse=8))
    assert e.value.code == lbm.EINVAL
    # a level-1 cell split although its level-2 parent is not: not a quadtree
    cfg = lbm.make_config(lattice=9, depth=2, nx_coarse=8, ny_coarse=8)
    with pytest.raises(lbm.LbmError) as e:
        lbm.Grid(cfg, split=[None, np.array([[4, 4]], np.int32), None])
    assert e.value.code == lbm.EMESH
    # two interfaces with no room for the ghost band between them (every child of the level-2 patch split again)
    s2 = np.array([[x, y] for x in range(2, 6) for y in range(2, 6)], np.int32)
    s1 = np.array([[x, y] for x in range(4, 12) for y in range(4, 12)], np.int32)
    with pytest.raises(lbm.LbmError) as e:
        lbm.Grid(cfg, split=[None, s1, s2])
    assert e.value.code == lbm.EMESH
    with pytest.raises(RuntimeError):
        O.OracleGrid(O.make_config(lattice=9, depth=2, nx_coarse=8, ny_coarse=8), [None, s1, s2])


def test_compute_calls_fail_loudly_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    g = lbm.Grid.from_case(W.tgv(16))
    with pytest.raises(lbm.LbmError) as e:
        g.bind()
    assert e.value.code == lbm.ECUDA
    z = np.zeros(g.ntot)
    assert g.init_fields(z + 1, z, z) == lbm.ESTATE      # not bound: no silent CPU path
    with pytest.raises(lbm.LbmError):
        g.step(1)
    g.close()


def test_matrix_addressing_is_refused_where_it_does_not_apply():
    """LBM_ADDR_MATRIX: single-level boxes without solids, weakly compressible models, periodic / wall sides only."""
    from paper_2504_04465_b200 import lbm
    ok = lbm.Grid.from_case(W.tgv(32), addressing=lbm.ADDR_MATRIX)
    ok.close()
    for case in (W.cavity(0.25), W.riemann(n=32), W.sod(L=32, lattice=13), W.cylinder(D=40, depth=3, radii=(3, 5, 8))):
        with pytest.raises(lbm.LbmError) as e:
            lbm.Grid.from_case(case, addressing=lbm.ADDR_MATRIX)
        assert e.value.code == lbm.EINVAL


def test_device_options_are_validated():
    """lbm_config.addressing / pipeline / pipe_max_ctas outside their ranges: LBM_EINVAL, no grid."""
    from paper_2504_04465_b200 import lbm
    case = W.tgv(16)
    for bad in (dict(addressing=7), dict(addressing=-1), dict(pipeline=3), dict(pipe_max_ctas=-2)):
        with pytest.raises(lbm.LbmError) as e:
            lbm.Grid.from_case(case, **bad)
        assert e.value.code == lbm.EINVAL
