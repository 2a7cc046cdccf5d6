"""GPU parity of the matrix-like uniform path (csrc/matrix.cuh; lbm_config.addressing = LBM_ADDR_MATRIX: Cartesian-index
addressing, AA-pattern in-place streaming, ONE population copy) against the oracle, which knows nothing of it: the
canonical post-collision state is read back through lbm_get_populations after EVEN and ODD numbers of steps (the two
storage layouts of the AA pattern), on periodic boxes (all four lattices, BGK and RR, non-square, sizes that are no
multiple of the CTA width), on the lid-driven cavity (bounce-back walls, moving lid: Ladd's term folded into the stored
values) and with a wall-normal inflow; plus the I/O round trip and the arena size."""
import numpy as np
import pytest

from helpers import gpu_from_case, max_pop_diff, oracle_from_case, rel_linf
from paper_2504_04465_b200 import lbm, workloads as W

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5}


def _periodic_case(nx, ny, lattice, collision):
    kx, ky = 2 * np.pi / nx, 2 * np.pi / ny

    def fields(level, ix, iy):
        x, y = W.centres(level, ix, iy)
        return (1.0 + 0.04 * np.sin(kx * x) * np.cos(2 * ky * y), 0.05 * np.sin(ky * y + 0.4) + 0.01,
                -0.04 * np.cos(kx * x) + 0.02, np.full(len(x), W.CS2[lattice]))
    return W.Case("box", W.uniform_mesh(nx, ny), lattice=lattice, collision=collision, tau0=0.63, fields=fields)


CASES = {
    "tgv64_q9_bgk": lambda: W.tgv(64),
    "box_150x70_q9_rr": lambda: _periodic_case(150, 70, 9, W.RR),
    "box_75x36_q9_bgk": lambda: _periodic_case(75, 36, 9, W.BGK),          # odd width: the one-cell-per-thread kernels
    "cavity_77_q13": lambda: W.cavity_uniform(77, lattice=13),
    "box_72x40_q13_rr": lambda: _periodic_case(72, 40, 13, W.RR),
    "box_48x56_q21_bgk": lambda: _periodic_case(48, 56, 21, W.BGK),
    "box_40x40_q37_rr": lambda: _periodic_case(40, 40, 37, W.RR),
    "cavity_96": lambda: W.cavity_uniform(96),
    "cavity_80_inflow": lambda: W.cavity_uniform(80, inflow=0.03),
    "cavity_64_q21": lambda: W.cavity_uniform(64, lattice=21, collision=W.BGK),
}


@pytest.mark.parametrize("name", sorted(CASES))
def test_matrix_path_matches_the_oracle_in_both_layouts(name):
    case = CASES[name]()
    precisions = (64, 32) if (case.lattice, 32, case.collision, 0, 0) in lbm.supported_models() else (64,)
    o = oracle_from_case(case)
    grids = {p: gpu_from_case(case, p, addressing=lbm.ADDR_MATRIX) for p in precisions}
    for g in grids.values():
        assert "matrix_step_kernel" in g.kernel_name()
        d0 = max_pop_diff(g, o)                       # initial state, layout P0
        assert d0 <= TOL[64 if g.cfg.precision == 64 else 32], (name, "init", d0)
    done = 0
    for upto in (1, 2, 7, 20):                        # odd and even step counts
        assert o.step(upto - done) == 0
        for p, g in grids.items():
            g.step(upto - done)
            assert g.sync() == 0
            d = max_pop_diff(g, o)
            assert d <= TOL[p] * (1 if upto <= 2 else 4), (name, p, upto, d)
        done = upto
    r, u, v, _ = o.macroscopic()
    for p, g in grids.items():
        gr, gu, gv, _ = g.macroscopic()
        tol = 1e-9 if p == 64 else 1e-4
        assert rel_linf(gr, r) <= tol and np.abs(gu - u).max() <= tol and np.abs(gv - v).max() <= tol, (name, p)
        g.close()


@pytest.mark.parametrize("n,lattice", [(79, 13), (97, 21), (130, 13), (61, 9)])
def test_matrix_lid_term_is_formed_by_the_owning_thread(n, lattice):
    """Ladd's term needs rho_w = sum_k S_k of the wall cell; in an odd AA step that cell's slots are overwritten by its
    neighbours, so the term must be folded in when the state is written (a version that summed the slots at reading time
    passed or failed with the launch timing).  Many steps, several widths, repeated: the result is the oracle's and the
    same in every run."""
    case = W.cavity_uniform(n, lattice=lattice, collision=W.BGK if lattice == 21 else W.RR)
    o = oracle_from_case(case)
    assert o.step(41) == 0
    ref = None
    for rep in range(3):
        g = gpu_from_case(case, 64, addressing=lbm.ADDR_MATRIX)
        for _ in range(41):
            g.step(1)
        assert g.sync() == 0
        S = g.populations(0)
        assert np.abs(S - o.populations(0)).max() <= 4e-12
        if ref is not None:
            assert np.array_equal(S, ref)
        ref = S
        g.close()


def test_matrix_path_1000_steps_cavity_and_probe_cells():
    case = W.cavity_uniform(64)
    o = oracle_from_case(case)
    g = gpu_from_case(case, 64, addressing=lbm.ADDR_MATRIX)
    assert o.step(1001) == 0
    g.step(1001)
    assert g.sync() == 0
    r, u, v, _ = o.macroscopic()
    gr, gu, gv, _ = g.macroscopic()
    assert rel_linf(gr, r) <= 1e-9 and np.abs(gu - u).max() <= 1e-9 * 0.1 + 1e-12 and np.abs(gv - v).max() <= 1e-10
    cells = np.array([0, 17, 4095, 2048, 63], np.int32)
    pr, pu, pv, _ = g.macroscopic_at(0, cells)
    assert np.array_equal(pr, gr[cells]) and np.array_equal(pu, gu[cells]) and np.array_equal(pv, gv[cells])
    g.close()


@pytest.mark.parametrize("steps_before", [0, 1])
def test_matrix_population_round_trip_and_restart(steps_before):
    """set_populations(get_populations()) leaves the run unchanged in either layout; a state imported from the tree-stored
    path continues identically (to rounding) on the matrix path."""
    case = CASES["cavity_96"]()
    a = gpu_from_case(case, 64, addressing=lbm.ADDR_MATRIX)
    b = gpu_from_case(case, 64, addressing=lbm.ADDR_LIST)
    a.step(4 + steps_before); b.step(4 + steps_before)
    assert a.sync() == 0 and b.sync() == 0
    S = a.populations(0)
    assert np.abs(S - b.populations(0)).max() <= 1e-13
    a.set_populations(0, 0, S)
    assert np.abs(a.populations(0) - S).max() <= 1e-15
    a.step(3); b.step(3)
    assert np.abs(a.populations(0) - b.populations(0)).max() <= 1e-13
    a.close(); b.close()


def test_matrix_arena_is_one_population_copy_and_no_tables():
    case = W.tgv(512)
    m = lbm.Grid.from_case(case, addressing=lbm.ADDR_MATRIX)
    t = lbm.Grid.from_case(case, addressing=lbm.ADDR_LIST)
    n = 512 * 512
    assert m.info.arena_bytes < 0.62 * t.info.arena_bytes
    assert m.info.arena_bytes <= n * (9 * 8 + 4 + 9 * 8) + 4096      # populations + order map + I/O scratch
    m.close(); t.close()


def test_matrix_path_follows_the_viscosity_and_lid_ramps_and_refuses_transfer():
    """lbm_set_relaxation / lbm_set_boundary_state between steps (the start-up ramps) on the matrix-like path against
    the oracle's setters, with single fine steps in between; lbm_transfer does not apply to it."""
    case = W.cavity_uniform(72)
    o = oracle_from_case(case)
    g = gpu_from_case(case, 64, addressing=lbm.ADDR_MATRIX)
    tau0 = case.tau0
    for step in range(6):
        t = W.viscosity_ramp_tau0(tau0, step, 5, factor=20.0)
        lid = 0.1 * W.mach_ramp_factor(step, 5)
        g.set_tau0(t); assert o.set_tau0(t) == 0
        g.set_bc_state(3, 1.0, lid, 0.0); assert o.set_bc_state(3, 1.0, lid, 0.0) == 0
        if step % 2:
            g.step_fine(3); assert o.step_fine(3) == 0
        else:
            g.step(2); assert o.step(2) == 0
        assert g.sync() == 0
    assert max_pop_diff(g, o) <= 4e-12
    other = gpu_from_case(W.cavity_uniform(72), 64, init=False)
    with pytest.raises(lbm.LbmError) as e:
        other.transfer_from(g)
    assert e.value.code == lbm.EINVAL
    g.close(); other.close()
