"""Pins of oracle_mapq_filter (next row f1: repeat filter + MAPQ), -m "not gpu".

The oracle computes MAPQ = -100 log2(second/best) with the C library's log2.  It is pinned here without log2: by the
numbers the paper prints (ratio .9 <-> 15.2, threshold 62), by closed forms at ratios 2^-k, by the inverse relation
second = best * 2^(-MAPQ/100) evaluated with exact rational / integer-power arithmetic, by monotonicity, and by the edge
readings (reading 17)."""
import os
from fractions import Fraction

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_constants.txt")


def _gold():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        out[k] = v
    return out


def _rec(best, second, bf=3, sf=5):
    return [[bf, 1, best, 0], [sf, 2, second, 1]]


def test_paper_printed_pair_ratio_09_is_152(oracle_mod):
    g = _gold()
    ratio, thr = Fraction(g["mapq_ratio"][0]), float(g["mapq_threshold"][0])       # .9 and 15.2
    recs = np.array([_rec(10 * k, int(10 * k * ratio)) for k in (1, 5, 10, 100, 3000)], dtype=np.int32)
    mapped, q = oracle_mod.mapq_filter(recs)
    assert (np.round(q, 1) == thr).all()                  # "-100 log2 .9 = 15.2" as printed, one decimal
    assert (mapped == 0).all()                            # mapped iff the ratio is BELOW .9
    # the literal printed cutoff 15.2 is a rounded value: as a MAPQ threshold it lets exactly .9 through, which is why
    # the default (threshold < 0) is decided on the integers
    assert (oracle_mod.mapq_filter(recs, thr)[0] == 1).all()
    assert (q > thr).all() and (q < thr + 1e-3).all()


def test_default_rule_is_exact_rational_comparison(oracle_mod):
    rng = np.random.default_rng(5701)
    best = rng.integers(1, 32768, size=4000)
    second = np.minimum(best, rng.integers(0, 32768, size=4000))
    near = rng.integers(1, 3276, size=2000)               # pairs on and next to the 9/10 boundary
    best = np.concatenate([best, 10 * near, 10 * near, 10 * near])
    second = np.concatenate([second, 9 * near, 9 * near - 1, 9 * near + 1])
    recs = np.array([_rec(int(b), int(s)) for b, s in zip(best, second)], dtype=np.int32)
    mapped, _ = oracle_mod.mapq_filter(recs)
    want = np.array([Fraction(int(s), int(b)) < Fraction(9, 10) for b, s in zip(best, second)], dtype=np.uint8)
    assert (mapped == want).all()


def test_closed_forms_powers_of_two(oracle_mod):
    # second/best = 2^-k  =>  MAPQ = 100 k exactly (log2 of a power of two is exact)
    recs = np.array([_rec(1 << 14, (1 << 14) >> k) for k in range(0, 15)], dtype=np.int32)
    _, q = oracle_mod.mapq_filter(recs)
    assert (q == 100.0 * np.arange(15)).all()
    # equal scores: p = 1, MAPQ = 0, never mapped under any threshold >= 0 or the default
    assert oracle_mod.mapq_filter(recs[:1])[0][0] == 0 and oracle_mod.mapq_filter(recs[:1], 0.0)[0][0] == 0


def test_inverse_relation_without_log(oracle_mod):
    """2^(-MAPQ/100) * best == second, checked through integer powers: (second/best)^100 == 2^(-MAPQ) within 1e-9 relative
    (exact rational left side, so a wrong base, sign or factor in the oracle's formula fails)."""
    rng = np.random.default_rng(5702)
    best = rng.integers(2, 32768, size=300)
    second = np.array([rng.integers(1, b + 1) for b in best])
    recs = np.array([_rec(int(b), int(s)) for b, s in zip(best, second)], dtype=np.int32)
    _, q = oracle_mod.mapq_filter(recs)
    for b, s, qq in zip(best, second, q):
        lhs = Fraction(int(s), int(b)) ** 100             # exact
        rhs = 2.0 ** (-qq)                                # one power of two of the reported value
        if rhs > 1e-300:
            assert abs(float(lhs) / rhs - 1.0) < 1e-9, (b, s, qq)
    # monotone: for a fixed best, MAPQ strictly falls as second grows
    recs = np.array([_rec(1000, s) for s in range(1, 1001)], dtype=np.int32)
    _, q = oracle_mod.mapq_filter(recs)
    assert (np.diff(q) < 0).all() and q[-1] == 0.0


def test_strict_threshold_62(oracle_mod):
    g = _gold()
    thr = float(g["mapq_threshold_strict"][0])
    # 62 <=> ratio < 2^-0.62; 2^-0.62 lies strictly between 650/1000 and 651/1000:
    # (650/1000)^100 < 2^-62 < (651/1000)^100 in exact rational arithmetic
    assert Fraction(650, 1000) ** 100 < Fraction(1, 2 ** 62) < Fraction(651, 1000) ** 100
    recs = np.array([_rec(1000, 650), _rec(1000, 651), _rec(2000, 1300), _rec(2000, 1302), _rec(100, 0)], dtype=np.int32)
    mapped, q = oracle_mod.mapq_filter(recs, thr)
    assert mapped.tolist() == [1, 0, 1, 0, 1]
    assert q[0] > thr > q[1]


def test_edge_readings(oracle_mod):
    recs = np.array([
        [[-1, 0, 0, 0], [-1, 0, 0, 0]],        # no fragment at all (bad read length): unmapped, MAPQ 0
        [[0, 0, 0, 0], [1, 0, 0, 0]],          # best = 0: the ratio is undefined -> unmapped (reading 17)
        [[4, 7, 120, 1], [-1, 0, 0, 0]],       # a genome of one fragment: no second place -> p = 0 -> mapped, MAPQ = +inf
        [[4, 7, 120, 0], [9, 3, 0, 0]],        # second fragment exists but scores 0 -> p = 0 -> mapped
        [[4, 7, 120, 0], [9, 3, 120, 1]],      # tie -> p = 1 -> MAPQ 0 -> unmapped
        [[4, 7, 1, 0], [9, 3, 0, 0]],          # smallest positive best
    ], dtype=np.int32)
    for thr in (-1.0, 15.2, 62.0, 0.0):
        mapped, q = oracle_mod.mapq_filter(recs, thr)
        assert mapped.tolist() == [0, 0, 1, 1, 0, 1]
        assert q[0] == 0.0 and q[1] == 0.0 and np.isinf(q[2]) and np.isinf(q[3]) and q[4] == 0.0 and np.isinf(q[5])
    # strand and window start never matter
    a = np.array([_rec(200, 130)], dtype=np.int32); b = a.copy(); b[0, :, 1] = 999; b[0, :, 3] = 1
    assert oracle_mod.mapq_filter(a)[1][0] == oracle_mod.mapq_filter(b)[1][0]


def test_builds_agree(oracle_mod):
    rng = np.random.default_rng(5703)
    best = rng.integers(0, 700, size=2000); second = np.minimum(best, rng.integers(0, 700, size=2000))
    recs = np.array([_rec(int(b), int(s), sf=int(rng.integers(-1, 3))) for b, s in zip(best, second)], dtype=np.int32)
    for thr in (-1.0, 15.2, 62.0):
        m2, q2 = oracle_mod.mapq_filter(recs, thr, opt="O2")
        m3, q3 = oracle_mod.mapq_filter(recs, thr, opt="O3")
        assert (m2 == m3).all() and np.array_equal(q2, q3)
