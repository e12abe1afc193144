"""Pins for the oracle's chunk table (Eq. 3, Table 8) and time model (Eq. 9-11, Tables 12-13).
CPU only.  Expected values come from tests/golden (typed from the paper) or from algebra."""
import math

import pytest

from oracle import hcms_oracle as O


def test_table8_chunk_lists_and_imbalance(golden_rows):
    # PAPER.md Table 8: H_per_rank = 10
    for C, sizes, imb in golden_rows("table8_chunks.txt"):
        sizes = [int(x) for x in sizes.split()]
        tab = O.chunk_table(10, int(C))
        assert [h for _, h in tab] == sizes
        assert round(100 * O.imbalance(sizes)) == int(imb)


@pytest.mark.parametrize("Hl", range(1, 41))
def test_chunk_table_invariants(Hl):
    for C in range(1, Hl + 1):
        tab = O.chunk_table(Hl, C)
        hs = [h for _, h in tab]
        assert sum(hs) == Hl                      # Eq. 3: H = sum H_c
        assert all(h >= 1 for h in hs)
        assert hs == sorted(hs, reverse=True)     # "more-first-less-later" L221
        assert max(hs) - min(hs) <= 1
        assert [o for o, _ in tab] == [sum(hs[:c]) for c in range(C)]   # Eq. 4 concat order
        assert hs.count(max(hs)) == (Hl % C or C)


def test_baseline_config_splits():
    # BASELINE.json configs state these per-rank splits
    assert [h for _, h in O.chunk_table(3, 2)] == [2, 1]          # cfg 2
    assert [h for _, h in O.chunk_table(10, 4)] == [3, 3, 2, 2]   # cfg 3
    assert [h for _, h in O.chunk_table(5, 2)] == [3, 2]          # cfg 4
    assert [h for _, h in O.chunk_table(3, 3)] == [1, 1, 1]       # cfg 5


@pytest.mark.parametrize("Hl,C", [(0, 1), (4, 0), (4, 5), (3, -1)])
def test_chunk_table_rejects(Hl, C):
    with pytest.raises(ValueError):
        O.chunk_table(Hl, C)


def test_table13_smax(golden_rows):
    for rho, printed in golden_rows("table13_smax.txt"):
        assert round(O.s_max(float(rho) / 100), 2) == float(printed)


def test_table12_cstar_row1(golden_rows):
    for rho, beta, t_total, pred in golden_rows("table12_cstar.txt"):
        t_comm = float(rho) / 100 * float(t_total)     # rho = T_comm / T_total (L154)
        cs = O.c_star(t_comm, float(beta))
        assert round(cs) == int(pred)
        assert abs(cs - 4.54) < 0.01                    # sqrt(29.03/1.41)


def test_eq11_is_eq9_over_eq10():
    # Eq. 11 must be T_base / T_hcms(C) with rho = T_comm/T_base (A.4, L425-427)
    for (t0, tc, ta, beta) in [(3.0, 29.0, 41.3, 1.41), (0.0, 10.0, 90.0, 0.0), (5.0, 1.0, 2.0, 0.3)]:
        tb = O.t_base(t0, tc, ta)
        assert tb == t0 + tc + ta
        for C in range(1, 12):
            th = O.t_hcms(C, t0, tc, ta, beta)
            assert math.isclose(O.speedup(C, tc / tb, beta, tb), tb / th, rel_tol=1e-13)


def test_time_model_limits_and_optimum():
    t0, tc, ta, beta = 2.0, 29.0, 40.0, 1.41
    # C = 1 with beta = 0 is the baseline (Eq. 9 == Eq. 10)
    assert O.t_hcms(1, t0, tc, ta, 0.0) == O.t_base(t0, tc, ta)
    # Theorem 2: beta -> 0, C -> inf gives 1/(1-rho)
    tb = O.t_base(t0, tc, ta)
    assert math.isclose(O.speedup(10**9, tc / tb, 0.0, tb), O.s_max(tc / tb), rel_tol=1e-8)
    # Theorem 1: C* minimises Eq. 10 over the reals => integer neighbours bracket it
    cs = O.c_star(tc, beta)
    best = min(range(1, 40), key=lambda C: O.t_hcms(C, t0, tc, ta, beta))
    assert best in (math.floor(cs), math.ceil(cs))
    eps = 1e-4
    f = lambda C: O.t_hcms(C, t0, tc, ta, beta)
    assert f(cs) <= f(cs - eps) and f(cs) <= f(cs + eps)


def test_choose_chunks_brute_force_agrees_with_theorem1(golden_rows):
    # Table 12 row 1 (L440): 40 heads on 8 GPUs = 5 per rank, C* = 4.54 -> the paper prints 5
    for rho, beta, t_total, pred in golden_rows("table12_cstar.txt"):
        assert O.choose_chunks(5, float(rho) / 100 * float(t_total), float(beta)) == int(pred)
    # unconstrained, the integer optimum is a neighbour of Theorem 1's C*; constrained, it is clamped
    for tc, beta in [(29.0, 1.41), (63.7, 6.83), (0.5, 0.004), (100.0, 0.01), (1.0, 5.0)]:
        cs = O.c_star(tc, beta)
        assert O.choose_chunks(10**4, tc, beta) in (max(1, math.floor(cs)), math.ceil(cs))
        assert O.choose_chunks(3, tc, beta) == min(3, O.choose_chunks(10**4, tc, beta))
    assert O.choose_chunks(7, 10.0, 0.0) == 7          # no per-chunk overhead: as many chunks as heads
