"""Test helpers: build an oracle simulation from a workloads.Case (test infrastructure)."""
import numpy as np

from oracle import oracle as O
from paper_2504_04465_b200 import workloads as W


def oracle_from_case(case, init=True):
    cfg = O.make_config(**case.model_kwargs())
    g = O.OracleGrid(cfg, case.mesh.split, case.mesh.solid)
    if init:
        cells = [g.cells(l)[:2] for l in range(g.depth + 1)]
        rho, ux, uy, T = W.eval_fields(case, cells)
        rc = g.init_fields(rho, ux, uy, T)
        assert rc == 0, "oracle init status %d" % rc
    return g


def level_slices(g):
    return [slice(int(g.off[l]), int(g.off[l + 1])) for l in range(g.depth + 1)]


def conserved_sums(g, Q_cx=None, Q_cy=None):
    """Mass and momentum (and population energy) over non-fine-ghost, in-box cells, weighted by cell area 4^l."""
    cx, cy, w, opp, cs2, reach = O.lattice(g.Q)
    M = PX = PY = E = 0.0
    for l in range(g.depth + 1):
        ix, iy, ty, aux = g.cells(l)
        keep = (ty == O.FLUID) | (ty == O.COARSE_GHOST)
        f = g.populations(l, 0)[keep]
        a = 4.0 ** l
        M += a * f.sum()
        PX += a * (f * cx).sum()
        PY += a * (f * cy).sum()
        e = (f * (cx * cx + cy * cy)).sum()
        if g.cfg.ddf:
            e += g.populations(l, 1)[keep].sum()
        E += a * e
    return np.array([M, PX, PY, E])


def gpu_from_case(case, precision=64, init=True, **device_options):
    """CUDA-path simulation of the same Case through the C ABI (tests marked gpu); device_options: lbm_config.addressing, ..."""
    from paper_2504_04465_b200 import lbm
    g = lbm.Grid.from_case(case, precision=precision, **device_options)
    g.bind()
    if init:
        cells = [g.cells(l)[:2] for l in range(g.depth + 1)]
        rho, ux, uy, T = W.eval_fields(case, cells)
        rc = g.init_fields(rho, ux, uy, T)
        assert rc == 0, "lbm_init_fields status %d" % rc
    return g


def max_pop_diff(g, o, which=(0,)):
    """max over levels, cells and components of |S_gpu - S_oracle| (ghost cells included)."""
    d = 0.0
    for l in range(o.depth + 1):
        if o.n[l] == 0:
            continue
        for w in which:
            d = max(d, float(np.abs(g.populations(l, w) - o.populations(l, w)).max()))
    return d


def rel_linf(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))
