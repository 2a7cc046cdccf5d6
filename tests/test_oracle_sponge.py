"""Pins of the pressure-relaxation sponge of the ORACLE (Eq. 10-11; reading S24 of DESIGN.md): the coefficient
field against its closed form, the no-op at p = p_inf, and the geometric relaxation rho_n - rho_inf = (1 - sigma)^n
(rho_0 - rho_inf) of a uniform state at unchanged velocity (streaming is the identity on a uniform periodic field and the
collision keeps rho and u, so the sponge is the only thing acting)."""
import numpy as np
import pytest

from helpers import oracle_from_case
from oracle import oracle as O
from paper_2504_04465_b200 import workloads as W


def uniform_case(n, rho, ux, uy, sponge, collision=W.RR, lattice=9):
    def fields(level, ix, iy):
        o = np.ones(len(ix))
        return rho * o, ux * o, uy * o, W.CS2[lattice] * o
    return W.Case("uniform", W.uniform_mesh(n, n), lattice=lattice, collision=collision, tau0=0.7, bc=(W.BC_PERIODIC,) * 4,
                  fields=fields, sponge=sponge)


def test_sigma_field_is_the_linear_ramp_of_eq11():
    case = W.cylinder(D=40, depth=3, radii=(3, 5, 8), sponge_d=(24, 30, 0.1))
    o = oracle_from_case(case, init=False)
    x0, y0, r0, r1, smax, _ = case.sponge
    seen = set()
    for l in range(o.depth + 1):
        ix, iy, ty, aux = o.cells(l)
        x, y = W.centres(l, ix, iy)
        r = np.hypot(x - x0, y - y0)
        expect = np.where(r >= r1, smax, np.where(r >= r0, smax * (r - r0) / (r1 - r0), 0.0))
        s = o.sponge(l)
        assert np.abs(s - expect).max() < 1e-14
        seen |= {("zero", bool((s == 0).any())), ("ramp", bool(((s > 0) & (s < smax)).any())), ("max", bool((s == smax).any()))}
    assert {("zero", True), ("ramp", True), ("max", True)} <= seen


@pytest.mark.parametrize("collision", [W.BGK, W.RR])
@pytest.mark.parametrize("lattice", [9, 13])
def test_uniform_state_relaxes_geometrically_at_constant_velocity(collision, lattice):
    sigma, rho_inf, rho0, ux, uy = 0.1, 1.0, 1.2, 0.05, -0.02
    o = oracle_from_case(uniform_case(16, rho0, ux, uy, (8.0, 8.0, 1e-9, 2e-9, sigma, rho_inf), collision, lattice))
    for n in range(1, 11):
        assert o.step(1) == 0
        r, u, v, T = o.macroscopic()
        assert np.abs(r - (rho_inf + (1 - sigma) ** n * (rho0 - rho_inf))).max() < 1e-13
        assert np.abs(u - ux).max() < 1e-14 and np.abs(v - uy).max() < 1e-14


def test_sponge_is_a_no_op_at_the_free_stream_pressure_and_rejects_thermal_models():
    sp = (8.0, 8.0, 1e-9, 2e-9, 0.1, 1.0)
    a = oracle_from_case(uniform_case(16, 1.0, 0.05, 0.0, sp))
    b = oracle_from_case(uniform_case(16, 1.0, 0.05, 0.0, None))
    assert a.step(5) == 0 and b.step(5) == 0
    assert np.abs(a.populations(0) - b.populations(0)).max() < 1e-15
    case = W.sod(L=16)
    case.sponge = sp
    with pytest.raises(Exception):
        O.OracleGrid(O.make_config(**case.model_kwargs()), case.mesh.split, case.mesh.solid)
