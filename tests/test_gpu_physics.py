"""A physical result of the CUDA path at scale against a value the PAPER prints (not against the oracle): the Strouhal
number of the vortex street behind the cylinder of configs[2] at (Re, Ma) = (150, 0.2), St = 0.1824 in the paper, 0.183 in
the DNS it cites, 0.179-0.185 in experiments (tests/golden/strouhal_aeolian.txt).  Half-resolution copy of the bench
workload (D = 100 finest cells, 6 levels, 2.5 M cells, inflow / Neumann / bounce-back links, every interface, the sponge of
Eq. 10-11) run for 400 convective times = 346 k fine steps (~25 s on a B200; the oracle would need a week), cross-stream
velocity probed two diameters behind the cylinder, spectrum by FFT with a Hamming window and zero padding as in P:317."""
import os

import numpy as np
import pytest

from paper_2504_04465_b200 import lbm, workloads as W

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "strouhal_aeolian.txt")


def test_cylinder_wake_strouhal_number_matches_the_paper():
    gold = {l.split()[0]: float(l.split()[1]) for l in open(GOLD) if l.strip() and not l.startswith("#")}
    D, every, t_total = 100, 8, 400.0
    case = W.cylinder(D=D, sponge_d=(24, 30, 0.1))
    g = lbm.Grid.from_case(case, precision=64).bind("cuda:0")
    cells = [g.cells(l)[:2] for l in range(g.depth + 1)]
    assert g.init_fields(*W.eval_fields(case, cells)) == 0
    u_inf = case.meta["u_inf"]
    tc = D / u_inf                                     # fine steps per convective time D / u_inf
    fine_per_coarse = 1 << g.depth
    ix, iy = cells[0]
    L = 64 * D
    probe = int(np.argmin((ix + 0.5 - (L / 2 + 2.0 * D)) ** 2 + (iy + 0.5 - L / 2) ** 2))
    t, v = [], []
    for s in range(0, int(t_total * tc / fine_per_coarse), every):
        g.step(every)
        v.append(g.macroscopic_at(0, [probe])[2][0])   # one probe cell, not the whole field
        t.append((s + every) * fine_per_coarse)
    assert g.sync() == 0                               # stable for 400 convective times
    g.close()
    t, v = np.array(t, float), np.array(v)
    n0 = int(0.6 * len(t))                             # the shedding has saturated by ~120 t_c
    sig = v[n0:] - v[n0:].mean()
    assert np.abs(sig).max() > 0.3 * u_inf             # a fully developed street: v' of the order of u_inf at the probe
    npad = 16 * len(sig)
    spec = np.abs(np.fft.rfft(sig * np.hamming(len(sig)), npad))
    freq = np.fft.rfftfreq(npad, d=t[1] - t[0])
    st = freq[spec[1:].argmax() + 1] * D / u_inf
    assert gold["experiment_lo"] <= st <= gold["experiment_hi"], st
    assert abs(st - gold["paper_lbm"]) < 0.003, st     # measured 0.1830 (fp64) / 0.1833 (fp32); DNS 0.183


@pytest.mark.parametrize("lattice,precision", [(13, 64), (21, 64), (37, 64), (21, 32)])
def test_sod_shock_tube_on_the_gpu_matches_the_exact_riemann_solution(lattice, precision):
    """The numerical-equilibrium + g + sensor kernels on the Sod tube of Eq. 12 at N = 1024 (an order of magnitude
    beyond what the oracle pin of tests/test_oracle_sod.py runs) against the exact solution of the Euler Riemann problem:
    first-order convergence carries the oracle's 0.9 % L1 density error at N = 256 down to ~0.25 %."""
    from test_oracle_sod import GAMMA, exact_riemann_density
    N = 1024
    case = W.sod(L=N, lattice=lattice, mesh="unif", periodic=False, ny=16)
    g = lbm.Grid.from_case(case, precision=precision).bind("cuda:0")
    cells = [g.cells(0)[:2]]
    assert g.init_fields(*W.eval_fields(case, cells)) == 0
    nsteps = int(round(0.2 * N / np.sqrt(GAMMA * W.SOD_T0[lattice])))
    g.step(nsteps)
    assert g.sync() == 0
    rho = g.macroscopic()[0]
    g.close()
    ix, iy = cells[0]
    m = (iy == 7) & (ix >= 0) & (ix < N)
    order = np.argsort(ix[m])
    x = ix[m][order] + 0.5
    (rl, _, Tl), (rr, _, Tr) = case.meta["left"], case.meta["right"]
    exact, _ = exact_riemann_density((x - N / 2) / nsteps, (rl, 0.0, rl * Tl), (rr, 0.0, rr * Tr))
    err = float(np.abs(rho[m][order] - exact).sum() / np.abs(exact).sum())
    assert err < 0.004, err


@pytest.mark.parametrize("lattice,collision", [(9, W.BGK), (9, W.RR), (13, W.RR), (21, W.RR), (37, W.RR)])
@pytest.mark.parametrize("precision", [64, 32])
def test_taylor_green_decay_rate_through_the_brick_path(lattice, collision, precision):
    """exp(-2 nu k^2 t) with nu = c_s^2 (tau - 1/2) (Eq. 3 / P6) on a 512^2 periodic box -- the smallest size that takes the
    regular-brick path by default (2^18 cells) -- for every weakly compressible lattice: the kinetic energy over 4000 steps
    decays at the analytic rate within the O(k^2) lattice error, in fp64 and in fp32."""
    n, steps = 512, 4000
    case = W.tgv(n, lattice=lattice, collision=collision)
    g = lbm.Grid.from_case(case, precision=precision).bind("cuda:0")
    assert "bricks" in g.kernel_name() and int(g.info.n_bricks[0]) * 64 == n * n
    cells = [g.cells(0)[:2]]
    assert g.init_fields(*W.eval_fields(case, cells)) == 0
    _, u0, v0, _ = g.macroscopic()
    g.step(steps)
    assert g.sync() == 0
    _, u1, v1, _ = g.macroscopic()
    g.close()
    m = case.meta
    rate = -np.log(np.sum(u1 ** 2 + v1 ** 2) / np.sum(u0 ** 2 + v0 ** 2)) / (2.0 * steps)       # energy decays twice as fast
    exact = 2.0 * m["nu"] * m["k"] ** 2
    assert abs(rate / exact - 1.0) < (2e-3 if precision == 64 else 2e-2), (rate, exact)


@pytest.mark.parametrize("lattice,collision", [(9, W.BGK), (13, W.RR), (21, W.RR), (37, W.RR)])
@pytest.mark.parametrize("precision", [64, 32])
def test_taylor_green_decay_rate_through_the_matrix_like_path(lattice, collision, precision):
    """The same physical law through the matrix-like path (Cartesian index, AA-pattern in-place streaming, one population copy):
    4001 steps (the state ends in the shifted layout), kinetic energy decays at exp(-4 nu k^2 t) within the O(k^2) lattice
    error; mass is conserved to accumulated rounding by the in-place update (4001 steps; D2Q37's 15-digit weights conserve
    to ~1e-14 per collision, S23)."""
    n, steps = 512, 4001
    case = W.tgv(n, lattice=lattice, collision=collision)
    g = lbm.Grid.from_case(case, precision=precision, addressing=lbm.ADDR_MATRIX).bind("cuda:0")
    assert "matrix_step_kernel" in g.kernel_name()
    cells = [g.cells(0)[:2]]
    assert g.init_fields(*W.eval_fields(case, cells)) == 0
    r0, u0, v0, _ = g.macroscopic()
    g.step(steps)
    assert g.sync() == 0
    r1, u1, v1, _ = g.macroscopic()
    g.close()
    m = case.meta
    rate = -np.log(np.sum(u1 ** 2 + v1 ** 2) / np.sum(u0 ** 2 + v0 ** 2)) / (2.0 * steps)
    exact = 2.0 * m["nu"] * m["k"] ** 2
    assert abs(rate / exact - 1.0) < (2e-3 if precision == 64 else 2e-2), (rate, exact)
    assert abs(r1.sum() / r0.sum() - 1.0) < (1e-9 if precision == 64 else 1e-3), r1.sum() / r0.sum() - 1.0
