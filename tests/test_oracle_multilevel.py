"""Pins for the oracle's multilevel part (DESIGN.md pins P8-P11): ghost band, unknown-direction masks,
coalescence / explosion (Eq. 4-5), asynchronous schedule (listing P:202-215)."""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2504_04465_b200 import workloads as W
from helpers import oracle_from_case, conserved_sums

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def smooth_fields(L, u0=0.03, rho_amp=0.02):
    """A smooth periodic low-Mach field on a box of L finest cells."""
    k = 2 * math.pi / L

    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        rho = 1.0 + rho_amp * np.sin(k * x) * np.cos(2 * k * y)
        ux = u0 * np.sin(k * y + 0.3) + 0.01
        uy = u0 * np.cos(2 * k * x) - 0.005
        return rho, ux, uy, np.full_like(x, 1.0 / 3.0)

    return fields


# ----------------------------------------------------------------------------- P11
def test_schedule_counts_and_order():
    case = W.patch(nc=64, lo=16, hi=48, depth=2, fields=smooth_fields(256))
    g = oracle_from_case(case)
    k, lv = g.schedule()
    seq = [[int(l) for l in lv[k == kk]] for kk in range(1, 5)]
    assert seq == [[0], [0, 1], [0], [0, 1, 2]]                   # canonical (pull) order, DESIGN.md
    for l in range(3):
        assert int((lv == l).sum()) == 2 ** (2 - l)               # n_t(i) = 2^(imax-i)
    # tau scaling, Eq. 3 with reading S3
    for l in range(3):
        assert g.tau(l) == pytest.approx(0.5 + (case.tau0 - 0.5) / 2 ** l, abs=1e-15)


def test_equivalent_fine_cells_table2():
    """'Equivalent fine cells' = sum_l N_l / 2^l reproduces the printed column of Table 2."""
    rows = []
    with open(os.path.join(GOLD, "table2_aeolian_grids.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            rows.append([int(t) for t in line.split()])
    assert len(rows) == 12
    for r in rows:
        levels, total, eq = r[1:-2], r[-2], r[-1]
        assert sum(levels) == total
        assert abs(sum(n / 2 ** l for l, n in enumerate(levels)) - eq) <= 1.0


# ----------------------------------------------------------------------------- structure of the ghost band
def test_ghost_band_structure_d2q9():
    case = W.patch(nc=32, lo=8, hi=24, depth=1, fields=smooth_fields(64))
    g = oracle_from_case(case)
    ix1, iy1, ty1, aux1 = g.cells(1)
    ix0, iy0, ty0, aux0 = g.cells(0)
    # coarse level: 32^2 - 16^2 unsplit cells; ghost ring = the 18^2 - 16^2 cells around the patch
    assert len(ix1) == 32 * 32 - 16 * 16
    assert int((ty1 == O.COARSE_GHOST).sum()) == 18 * 18 - 16 * 16
    # fine level: 32^2 bulk + 4 children per coarse ghost
    assert int((ty0 == O.FLUID).sum()) == 32 * 32
    assert int((ty0 == O.FINE_GHOST).sum()) == 4 * (18 * 18 - 16 * 16)
    co, ch, mask = g.ghosts(1)
    assert (ch >= 0).all()
    # Morton order with x in the even bits (reading S5)
    def morton(x, y):
        k = np.zeros(len(x), np.uint64)
        for b in range(16):
            k |= ((x.astype(np.uint64) >> np.uint64(b)) & np.uint64(1)) << np.uint64(2 * b)
            k |= ((y.astype(np.uint64) >> np.uint64(b)) & np.uint64(1)) << np.uint64(2 * b + 1)
        return k
    for ix, iy in ((ix0, iy0), (ix1, iy1)):
        key = morton(ix, iy)
        assert (np.diff(key.astype(np.int64)) > 0).all()
    # unknown directions of a coarse ghost = pull sources that are split cells
    cx, cy, w, opp, cs2, reach = O.lattice(9)
    nbr = g.nbr(1)
    for q in range(len(co)):
        c = co[q]
        for i in range(1, 9):
            sx, sy = ix1[c] - cx[i], iy1[c] - cy[i]
            split = 8 <= sx < 24 and 8 <= sy < 24
            assert bool((int(mask[q]) >> i) & 1) == split
            assert (nbr[c, i - 1] == O.LINK_NONE) == split
    # children are stored in order a + 2b
    for q in range(len(co)):
        c = co[q]
        for k in range(4):
            assert ix0[ch[q, k]] == 2 * ix1[c] + (k & 1) and iy0[ch[q, k]] == 2 * iy1[c] + (k >> 1)
            assert ty0[ch[q, k]] == O.FINE_GHOST


@pytest.mark.parametrize("Q,reach", [(9, 1), (13, 2), (21, 3), (37, 3)])
def test_ghost_band_width_high_order(Q, reach):
    """Buffer of 1 / 2 / 3 coarse layers for D2Q9 / D2Q13 / D2Q21, D2Q37 (Fig. 3)."""
    case = W.stripe(nc=32, lo=10, hi=22, lattice=Q, fields=smooth_fields(64))
    g = oracle_from_case(case, init=False)
    ix1, iy1, ty1, _ = g.cells(1)
    gx = np.unique(ix1[ty1 == O.COARSE_GHOST])
    expect = list(range(10 - reach, 10)) + list(range(22, 22 + reach))
    assert gx.tolist() == expect


def test_mesh_errors():
    # interface running into a Neumann side (ghost cells would need boundary-cell copies): rejected
    def refine(level, ix, iy):
        return iy < 4
    mesh = W.build_mesh(1, 16, 16, refine)
    cfg = O.make_config(lattice=9, depth=1, nx_coarse=16, ny_coarse=16, bc=(O.BC_NEUMANN, O.BC_NEUMANN, O.BC_PERIODIC, O.BC_PERIODIC))
    with pytest.raises(RuntimeError):
        O.OracleGrid(cfg, mesh.split, mesh.solid)
    # two interfaces without room for the ghost bands (level jump of 2): rejected
    def refine2(level, ix, iy):
        if level == 2:
            return (ix >= 4) & (ix < 12)
        return (ix >= 8) & (ix < 24)       # all children of the split level-2 cells
    mesh = W.build_mesh(2, 16, 16, refine2)
    cfg = O.make_config(lattice=9, depth=2, nx_coarse=16, ny_coarse=16)
    with pytest.raises(RuntimeError):
        O.OracleGrid(cfg, mesh.split, mesh.solid)


# ----------------------------------------------------------------------------- P8
@pytest.mark.parametrize("Q,coll", [(9, O.BGK), (9, O.RR), (13, O.RR), (21, O.BGK)])
def test_conservation_straight_interface(Q, coll):
    """Coalescence and explosion are conservative: on a periodic box with two straight interfaces
    mass and momentum over the non-ghost cells (weighted by cell area) stay constant to rounding."""
    case = W.stripe(nc=32, lo=10, hi=22, lattice=Q, collision=coll, tau0=0.7, fields=smooth_fields(64))
    g = oracle_from_case(case)
    s0 = conserved_sums(g)
    for _ in range(10):
        g.step(1)
        s = conserved_sums(g)
        assert abs(s[0] - s0[0]) <= 2e-13 * s0[0]
        assert abs(s[1] - s0[1]) <= 2e-13 * s0[0]
        assert abs(s[2] - s0[2]) <= 2e-13 * s0[0]


def test_conservation_patch_corner_leak_is_small():
    """With corners, fine bulk cells exchange diagonal populations with fine ghosts whose parent's same
    population travels coarse-to-coarse; the reading of P:112 ('unknown = not received from a coarse
    neighbour') then leaks O(gradient) mass at the four corners (reading S8b).  The drift is
    bounded and tiny; uniform states are preserved exactly (next test)."""
    case = W.patch(nc=32, lo=8, hi=24, depth=1, tau0=0.7, fields=smooth_fields(64))
    g = oracle_from_case(case)
    s0 = conserved_sums(g)
    g.step(20)
    s = conserved_sums(g)
    assert abs(s[0] - s0[0]) <= 1e-6 * s0[0]


@pytest.mark.parametrize("coll", [O.BGK, O.RR])
def test_uniform_flow_exact_across_interface(coll):
    """P10 (exact part): a uniform state is reproduced exactly across corners and staircases."""
    def fields(level, ix, iy):
        o = np.ones(len(ix))
        return 1.1 * o, 0.04 * o, -0.02 * o, o / 3
    case = W.patch(nc=32, lo=8, hi=24, depth=2, collision=coll, tau0=0.6, fields=fields)
    g = oracle_from_case(case)
    f0 = [g.populations(l).copy() for l in range(3)]
    g.step(3)
    for l in range(3):
        assert np.abs(g.populations(l) - f0[l]).max() < 5e-16


# ----------------------------------------------------------------------------- P9
def _feq_product_d2q9(rho, ux, uy, cx, cy):
    """Closed-form product equilibrium of the D2Q9 partial-4th-order expansion (pinned in test_oracle_physics P2)."""
    def phi(c, u):
        return np.where(c == 0, 2.0 / 3.0 - u * u, (1.0 + 3.0 * c * u + 3.0 * u * u) / 6.0)
    return rho[..., None] * phi(cx[None, None, :], ux[..., None]) * phi(cy[None, None, :], uy[..., None])


def _bgk(P, tau, cx, cy):
    rho = P.sum(-1)
    ux = (P * cx).sum(-1) / rho
    uy = (P * cy).sum(-1) / rho
    feq = _feq_product_d2q9(rho, ux, uy, cx, cy)
    return P - (P - feq) / tau


def test_pull_form_equals_paper_push_form():
    """P9: the oracle's canonical pull form with post-collision storage equals a literal transcription of
    the paper's listing (coupling, then collide-and-push, coarse level first, pre-collision
    storage) on a 16x16 two-level periodic box: S(t) = collide(P(t))."""
    nc, lo, hi, tau0 = 16, 5, 11, 0.8
    nf = 2 * nc
    cx, cy, w, opp, cs2, reach = O.lattice(9)
    fields = smooth_fields(nf)
    case = W.patch(nc=nc, lo=lo, hi=hi, depth=1, tau0=tau0, fields=fields)
    g = oracle_from_case(case)
    tau = [tau0, 0.5 + (tau0 - 0.5) / 2]

    # ---- literal push-form reference on dense arrays
    CX, CY = np.meshgrid(np.arange(nc), np.arange(nc), indexing="ij")     # arrays indexed [ix, iy]
    split = (CX >= lo) & (CX < hi) & (CY >= lo) & (CY < hi)
    near = np.zeros_like(split)
    for dx in (-1, 0, 1):
        for dy in (-1, 0, 1):
            near |= np.roll(np.roll(split, dx, 0), dy, 1)
    cghost = near & ~split
    FX, FY = np.meshgrid(np.arange(nf), np.arange(nf), indexing="ij")
    fbulk = split[FX // 2, FY // 2]
    fghost = cghost[FX // 2, FY // 2]
    fstored = fbulk | fghost

    def init(level, n):
        X, Y = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
        rho, ux, uy, _ = fields(level, X.ravel(), Y.ravel())
        return _feq_product_d2q9(rho.reshape(n, n), ux.reshape(n, n), uy.reshape(n, n), cx, cy)

    Pc, Pf = init(1, nc), init(0, nf)

    def coupling():
        for x, y in zip(*np.nonzero(cghost)):
            for i in range(1, 9):
                sx, sy = (x - cx[i]) % nc, (y - cy[i]) % nc
                if split[sx, sy]:                                  # did not receive a value from a coarse neighbour
                    Pc[x, y, i] = Pf[2 * x:2 * x + 2, 2 * y:2 * y + 2, i].sum() / 4.0     # Eq. 4
            post = _bgk(Pc[x:x + 1, y:y + 1], tau[1], cx, cy)[0, 0]
            Pf[2 * x:2 * x + 2, 2 * y:2 * y + 2, :] = post            # Eq. 5

    def collide_and_stream(P, stored, collide_mask, t, n):
        post = np.where(collide_mask[..., None], _bgk(P, t, cx, cy), P)
        new = P.copy()
        for i in range(9):
            shifted = np.roll(np.roll(post[..., i], cx[i], 0), cy[i], 1)        # push to x + xi_i
            src_ok = np.roll(np.roll(stored, cx[i], 0), cy[i], 1)
            new[..., i] = np.where(stored & src_ok, shifted, new[..., i])
        return new

    def compare(tag):
        coupling()                                                 # the coupling of the iteration about to start
        Sc = _bgk(Pc, tau[1], cx, cy)
        Sf = np.where(fbulk[..., None], _bgk(Pf, tau[0], cx, cy), Pf)
        ix1, iy1, ty1, _ = g.cells(1)
        ix0, iy0, ty0, _ = g.cells(0)
        d1 = np.abs(g.populations(1) - Sc[ix1, iy1]).max()
        d0 = np.abs(g.populations(0) - Sf[ix0, iy0]).max()
        assert d1 < 1e-14 and d0 < 1e-14, (tag, d0, d1)

    with np.errstate(invalid="ignore", divide="ignore"):           # unstored dense entries hold junk
        compare("t=0")
        # undo nothing: the reference's coupling of iteration 0 has just run; continue the listing from there
        it = 0
        for coarse_step in range(8):
            for sub in range(2):
                if it % 2 == 0 and it > 0:
                    pass                                           # coupling already applied by compare()
                if it % 2 == 0:
                    Pc = collide_and_stream(Pc, ~split, ~split, tau[1], nc)
                Pf = collide_and_stream(Pf, fstored, fbulk, tau[0], nf)
                it += 1
            g.step(1)
            compare("after coarse step %d" % (coarse_step + 1))


# ----------------------------------------------------------------------------- P10
def _run_case(case, coarse_steps):
    g = oracle_from_case(case)
    g.step(coarse_steps)
    return g


def test_multilevel_vs_uniform_fine_converges():
    """P10: multilevel and uniform-fine solutions of a smooth low-Mach flow differ by a few percent on a
    16^2 coarse box and the difference shrinks under refinement (diffusive scaling).  Uniform explosion is
    piecewise constant (no interpolation), so the interface is first-order: the observed factor is
    about 2 per doubling, not 4 (pin P10)."""
    errs = []
    for nc, tau0, steps_c in ((16, 0.8, 4), (32, 0.8, 16)):
        nf = 2 * nc
        u0 = 0.04 * 16 / nc                                        # diffusive scaling: Mach halves with dx
        k = 2 * math.pi / nf

        def fields(level, ix, iy, u0=u0, k=k):
            x, y = W.centres(level, ix, iy)
            ux = -u0 * np.cos(k * x) * np.sin(k * y)
            uy = u0 * np.sin(k * x) * np.cos(k * y)
            rho = 1.0 - (3 * u0 * u0 / 4) * (np.cos(2 * k * x) + np.cos(2 * k * y))
            return rho, ux, uy, np.full_like(x, 1 / 3)

        ml = _run_case(W.patch(nc=nc, lo=nc // 4, hi=3 * nc // 4, depth=1, tau0=tau0, fields=fields), steps_c)
        un = W.tgv(n=nf, tau=tau0)
        un.fields = fields
        uf = _run_case(un, 2 * steps_c)
        r, u, v, _ = uf.macroscopic()
        ixu, iyu, _, _ = uf.cells(0)
        dense_u = np.zeros((nf, nf)); dense_v = np.zeros((nf, nf))
        dense_u[ixu, iyu] = u; dense_v[ixu, iyu] = v
        rm, um, vm, _ = ml.macroscopic()
        ix0, iy0, ty0, _ = ml.cells(0)
        sl = slice(int(ml.off[0]), int(ml.off[1]))
        bulk = ty0 == O.FLUID
        e = np.sqrt(((um[sl][bulk] - dense_u[ix0[bulk], iy0[bulk]]) ** 2 + (vm[sl][bulk] - dense_v[ix0[bulk], iy0[bulk]]) ** 2).mean()) / u0
        errs.append(e)
    assert errs[0] < 0.05
    assert errs[1] < errs[0] / 1.6


def test_ramp_setters_follow_eq3_and_reject_bad_arguments():
    """orc_set_tau0: tau_l - 1/2 = (tau_0 - 1/2) / 2^l (Eq. 3, S3) on every level; tau_0 < 1/2 and a side outside 0..3 are
    rejected; the viscosity-ramp helper starts at 100 nu and ends at nu."""
    case = W.patch(nc=48, lo=8, hi=40, depth=2)
    o = oracle_from_case(case, init=False)
    assert o.set_tau0(0.9) == 0
    for l in range(3):
        assert o.tau(l) == pytest.approx(0.5 + 0.4 / 2 ** l, abs=1e-15)
    assert o.set_tau0(0.49) != 0 and o.set_bc_state(4, 1.0, 0.0, 0.0) != 0
    assert W.viscosity_ramp_tau0(0.6, 0, 10) == pytest.approx(0.5 + 0.1 * 100)
    assert W.viscosity_ramp_tau0(0.6, 10, 10) == pytest.approx(0.6) and W.viscosity_ramp_tau0(0.6, 25, 10) == pytest.approx(0.6)
    assert W.mach_ramp_factor(0, 4) == 0.5 and W.mach_ramp_factor(4, 4) == 1.0
