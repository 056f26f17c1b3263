"""Host logic of bench.py that needs no GPU: the rule that picks PDD's partitions (never by hand: reading A9 of DESIGN.md),
checked with the ORACLE's a-priori bound standing in for tdx_pdd_dropped_bound; the look-up of `roofline.traffic` in the
committed ncu table; the sample shapes of the cpu_baseline leg; the tuned table's validity as partition maps."""
import os
import sys

import numpy as np
import pytest

import oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_1812_01178_b200 import configs  # noqa: E402

BCS = (orc.BC_DIRICHLET, orc.BC_DIRICHLET, orc.BC_PERIODIC)


class OracleBoundGrid:
    """Stand-in for binding.Grid in bench.pdd_partitions: the a-priori PDD bound from the oracle's definition."""

    def __init__(self, cfg):
        self.faces = cfg.faces()
        self.calls = []

    def pdd_dropped_bound(self, direction, P, alpha):
        self.calls.append((direction, P))
        a, b, c = orc.adi_coeffs(self.faces[direction], BCS[direction], alpha)
        return orc.cyclic_pdd_dropped(P, a, b, c) if BCS[direction] == orc.BC_PERIODIC else orc.pdd_dropped(P, a, b, c)


@pytest.mark.parametrize("cfg_no", [1, 2, 3, 4, 5])
def test_pdd_partitions_rule_gives_a_gated_divisor_not_above_the_ppt_choice(cfg_no):
    cfg = configs.get(cfg_no)
    g = OracleBoundGrid(cfg)
    for direction in range(3):
        n = (cfg.nx, cfg.ny, cfg.nz)[direction]
        Pt = bench.TUNED_P[cfg_no][direction]
        P, bound = bench.pdd_partitions(g, cfg, direction, Pt)
        assert 1 <= P <= Pt and (P == 1 or (n % P == 0 or P == Pt)) and (P == 1 or n // P >= 2)
        if P > 1:
            assert bound <= bench.PDD_GATE
            a, b, c = orc.adi_coeffs(g.faces[direction], BCS[direction], cfg.alpha)
            want = orc.cyclic_pdd_dropped(P, a, b, c) if BCS[direction] == orc.BC_PERIODIC else orc.pdd_dropped(P, a, b, c)
            assert bound == want
        # every candidate the rule passed over on the way down was tried in order and failed the gate
        tried = [p for d, p in g.calls if d == direction]
        assert tried[0] == Pt and tried[-1] == P or P == 1
        for p in tried[:-1]:
            assert g.pdd_dropped_bound(direction, p, cfg.alpha) > bench.PDD_GATE


def test_pdd_partitions_on_the_gate_grids_are_the_documented_ones():
    """DESIGN.md reading A9 / README: cfg4 y -> 8 (PPT runs 32; 16 drops 3.6e-7), cfg5 y -> the PPT-tuned 12."""
    c4, c5 = configs.get(4), configs.get(5)
    assert bench.pdd_partitions(OracleBoundGrid(c4), c4, 1, bench.TUNED_P[4][1])[0] == 8
    assert bench.pdd_partitions(OracleBoundGrid(c4), c4, 1, 16)[0] == 8
    P5, b5 = bench.pdd_partitions(OracleBoundGrid(c5), c5, 1, bench.TUNED_P[5][1])
    assert P5 == bench.TUNED_P[5][1] == 12 and b5 < 1e-20
    assert bench.pdd_partitions(OracleBoundGrid(c5), c5, 1, 24)[0] == 18        # the round's earlier table: 24 -> 18


def test_tuned_table_holds_valid_partition_maps():
    for cfg_no, Ps in bench.TUNED_P.items():
        cfg = configs.get(cfg_no)
        for n, P in zip((cfg.nx, cfg.ny, cfg.nz, cfg.ny), Ps):
            assert 1 <= P <= 1024 and n // P >= 2, (cfg_no, n, P)
            st = orc.partition_bounds(n, P)
            assert st[0] == 0 and st[-1] == n and np.all(np.diff(st) >= 2)


def test_ncu_traffic_lookup_is_keyed_by_workload_and_launch_shape():
    import csv
    with open(bench.NCU_TRAFFIC_FILE) as f:
        rows = list(csv.DictReader(r for r in f if not r.startswith("#")))
    assert len(rows) >= 8
    for row in rows:
        cfg = configs.get(int(row["workload"][3]))
        got, src = bench.ncu_traffic(row["workload"], row["launch"])
        assert got == float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]) and "r2_ncu_traffic.csv" in src
        # a sweep moves its algorithmic 16 B per real value (32 B per complex Helmholtz value) and nothing more
        alg_field, alg_helm = 16.0 * cfg.npts, 32.0 * cfg.nx * cfg.ny * cfg.nm
        assert min(abs(got / alg_field - 1.0), abs(got / alg_helm - 1.0)) < 0.03, (row["launch"], got)
    w, l = rows[0]["workload"], rows[0]["launch"]
    assert bench.ncu_traffic(w, l.replace("block=(", "block=(1")) == (None, "no committed ncu capture for %s on %s" % (l.replace("block=(", "block=(1"), w))
    assert bench.ncu_traffic("cfg9_none", l)[0] is None                          # another workload: no figure


def test_cpu_baseline_sample_is_bounded_and_a_subset_of_the_workload():
    for cfg_no in (1, 2, 3, 4, 5, 6):
        cfg = configs.get(cfg_no)
        kx, jz, mh = bench.sample_shapes(cfg)
        assert 1 <= kx <= cfg.nz and 1 <= jz <= cfg.ny and 1 <= mh <= cfg.nm
        vals = 2 * kx * cfg.nx * cfg.ny + jz * cfg.nx * cfg.nz + 2 * mh * cfg.nx * cfg.ny       # real values of the sample
        assert vals <= 4 * 250_000_000 or (kx == 1 and jz == 1 and mh == 1)
    assert bench.step_points(configs.get(5)) == 3 * 4096 * 288 * 512 + 2 * 4096 * 288 * 257
