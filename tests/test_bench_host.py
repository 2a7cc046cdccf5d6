"""Host-side logic of bench.py for N > 1 (replicas only): max-over-ranks timing with world_size-2 gloo,
and the reference arm under torchrun (rank 0 alone prints, the other ranks exit 0 without work)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, e2e = bench.reduce_max_over_ranks([10.0 + 5.0 * rank, 100.0 - rank], world)
    q.put((rank, ms, e2e, bench.aggregate_mlups(1000, 4, world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for rank, ms, e2e, v in res:
        assert ms == 15.0 and e2e == 100.0          # every rank sees the slowest rank's time
        assert v == pytest.approx(1000 * 4 * 2 / 15e-3 / 1e6)


def test_reference_arm_under_torchrun_prints_one_line():
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "cavity",
           "--scale", "0.25", "--steps", "2", "--warmup", "1"]
    r = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["unit"] == "MLUPS"


def test_algorithmic_bytes_per_update_match_the_scope_table():
    """SURVEY 8(d) / DESIGN.md Sec. 11: 2*npop*s + (Q-1)*4 + 4 bytes per cell update of the list-addressed method."""
    import bench
    from paper_2504_04465_b200 import workloads as W
    assert bench.algorithmic_bytes_per_update(W.tgv(64), 64) == 180
    assert bench.algorithmic_bytes_per_update(W.tgv(64), 32) == 108
    assert bench.algorithmic_bytes_per_update(W.tgv(64, lattice=13, collision=W.RR), 64) == 260
    assert bench.algorithmic_bytes_per_update(W.tgv(64, lattice=21, collision=W.RR), 64) == 420
    assert bench.algorithmic_bytes_per_update(W.riemann(n=64), 64) == 1332
    assert bench.algorithmic_bytes_per_update(W.naca(chord=64, depth=3, radii=(1, 2.5, 5)), 64) == 884
    # Table 3a of the paper is carried verbatim
    assert bench.PAPER_TABLE3[(21, "unif")] == 618.5 and bench.PAPER_TABLE3[(37, "band")] == 307.4 and len(bench.PAPER_TABLE3) == 12


def test_moved_bytes_count_bricks_only_on_large_levels():
    """Bytes the implementation must move: a 64^2 box is below the 2^18-cell threshold (list: 2*9*8 + 32 + 1 B),
    a 1024^2 box is all bricks (144 B + 36 B per 64 cells)."""
    import bench
    from paper_2504_04465_b200 import lbm, workloads as W
    small = lbm.Grid.from_case(W.tgv(64))
    assert bench.moved_bytes_per_update(small, W.tgv(64), 64) == 2 * 9 * 8 + 32 + 1
    big = lbm.Grid.from_case(W.tgv(1024))
    assert bench.moved_bytes_per_update(big, W.tgv(1024), 64) == pytest.approx(144 + 36 / 64)
    small.close(); big.close()


def test_byte_accounting_reproduces_the_papers_list_penalty_table():
    """Eq. 14-16: a matrix-like update moves 2 n s + 8 B per cell, the tree adds (Q-1) 4 B of neighbour list; the
    ratios of Table 1 (golden fixture) follow, and bench.py's list-addressed figure is the tree's minus the 4 B own index that
    a pull kernel does not read."""
    import bench
    from paper_2504_04465_b200 import workloads as W
    gold = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "table1_list_penalty.txt")):
        if line.strip() and not line.startswith("#"):
            c = line.split()
            gold[(c[0], c[1])] = [float(x) for x in c[2:]]
    for (model, prec), ratios in gold.items():
        s = 4 if prec == "sp" else 8
        for Q, r in zip((9, 13, 21, 37), ratios):
            n = Q if model == "weakly" else 2 * Q + 8
            matrix, tree = 2 * n * s + 8, 2 * n * s + 8 + (Q - 1) * 4
            assert abs(matrix / tree - r) < 0.0051, (model, prec, Q, matrix / tree, r)
    for prec, s in ((64, 8), (32, 4)):
        assert bench.algorithmic_bytes_per_update(W.tgv(64), prec) == 2 * 9 * s + 8 + 8 * 4 - 4
    naca = W.naca(chord=64, depth=3, radii=(1, 2.5, 5))
    assert bench.algorithmic_bytes_per_update(naca, 64) == 2 * (2 * 21 + 8) * 8 + 8 + 20 * 4 - 4


def _bench():
    import bench
    return bench


def test_roofline_fraction_is_in_moved_bytes_and_flagged_when_implausible():
    """the headline fraction counts the bytes the kernel moves (a brick cell reads no list), so a kernel at copy
    speed reads ~1.0, and anything above 1.05 is flagged; the list-addressed figure of SURVEY 8(d) sits beside it."""
    import types
    from paper_2504_04465_b200 import workloads as W
    bench = _bench()
    case = W.tgv(1024)
    g = types.SimpleNamespace(depth=0, n=[1024 * 1024], kernel_name=lambda: "sweep_kernel<...> (bricks + list)",
                              info=types.SimpleNamespace(n_bricks=[1024 * 1024 // 64], brick_min_level_cells=1 << 18))
    mbpu = bench.moved_bytes_per_update(g, case, 64)
    assert abs(mbpu - (144 + 36.0 / 64)) < 1e-9
    peak = 6500.0
    hbm, alu = bench.roofline_blocks(case, 64, g, "none", 1.0, peak * 1e9 / mbpu, peak, "test", None)
    assert alu is None and abs(hbm["frac"] - 1.0) < 1e-12 and hbm["frac_plausible"]
    assert abs(hbm["list_addressed"]["frac"] - 180.0 / mbpu) < 1e-12 and hbm["list_addressed"]["frac"] > 1.2
    hbm, _ = bench.roofline_blocks(case, 64, g, "none", 1.0, 1.3 * peak * 1e9 / mbpu, peak, "test", None)
    assert not hbm["frac_plausible"]
    m = types.SimpleNamespace(depth=0, n=[1024 * 1024], kernel_name=lambda: "matrix_step_kernel<9,double,LBM_BGK> (Cartesian index, AA pattern)",
                              info=g.info)
    assert bench.moved_bytes_per_update(m, case, 64) == 144.0


def test_committed_bench_lines_have_plausible_fractions():
    """Every bench line kept under profiles/bench/ for this round: the HBM fraction (moved bytes / measured copy bandwidth) of
    the headline and of every `also` entry stays <= 1.05."""
    import glob
    import json
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "bench", "r02_*.txt")))
    for f in files:
        for line in open(f):
            if not line.startswith("{"):
                continue
            d = json.loads(line)
            for blk in [d] + d.get("also", []):
                r = blk.get("roofline_hbm") or blk.get("roofline")
                if r and r.get("bound") == "hbm":
                    assert r["frac"] <= 1.05, (f, blk.get("entry"), r["frac"])
