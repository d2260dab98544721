"""The inequality behind the two-pass scan, checked exhaustively on the CPU with no product code:
for every match/mismatch pattern of up to 13 scored positions and several (match, mismatch) pairs, the pass-1 recurrence
    G <- max(G + s1 + s2, 0) over consecutive pairs (a lone last position as G <- max(G + s1, 0)), Bt = max of the sampled G
satisfies  Bt <= best <= Bt + min(M, -X) - X  where best is the exact maximum scoring subsequence, here by brute
force over all sub-ranges.  The bound is also tight for 5/-4 (some pattern reaches the full slack)."""
import itertools

import pytest


def exact_best(scores):
    best = 0
    for a in range(len(scores)):
        tot = 0
        for b in range(a, len(scores)):
            tot += scores[b]
            best = max(best, tot)
    return best


def pass1_bound(scores):
    g = bt = 0
    for j in range(0, len(scores), 2):
        a = scores[j] + (scores[j + 1] if j + 1 < len(scores) else 0)
        g = max(g + a, 0)
        bt = max(bt, g)
    return bt


@pytest.mark.parametrize("M,X", [(5, -4), (1, -1), (2, -7), (9, -3), (3, -5), (10, -40), (4, -4)])
def test_bound_exhaustive(M, X):
    delta = min(M, -X) - X
    worst = 0
    for n in range(1, 14):
        for pat in itertools.product((M, X), repeat=n):
            best, bt = exact_best(pat), pass1_bound(pat)
            assert bt <= best <= bt + delta, (pat, best, bt)
            worst = max(worst, best - bt)
    assert worst <= delta
    if (M, X) == (5, -4):
        assert worst == delta          # the slack of 8 is reached: the bound cannot be tightened


def test_bound_position_specific_scores():
    """The same recurrence under base-quality scoring (PSSM form): every position i has its own
    pmatch_i in [0, PM] and pmismatch_i in [PMM, 0]; the slack is min(PM, -PMM) - PMM with PM / PMM the table's stated range.
    Exhaustive over match patterns of up to 10 positions for random tables (including the extreme values and zeros), and
    exhaustive over ALL tables with values in a small grid for up to 4 positions."""
    import random
    rng = random.Random(1403)
    for PM, PMM in ((80, -22), (5, -4), (40, -11), (7, -30), (16, -16)):
        delta = min(PM, -PMM) - PMM
        worst = 0
        for _ in range(60):
            n = rng.randint(1, 10)
            pm = [rng.choice((0, 1, PM // 2, PM - 1, PM)) for _ in range(n)]
            px = [rng.choice((0, -1, PMM // 2, PMM + 1, PMM)) for _ in range(n)]
            for pat in itertools.product((0, 1), repeat=n):
                s = [pm[i] if pat[i] else px[i] for i in range(n)]
                best, bt = exact_best(s), pass1_bound(s)
                assert bt <= best <= bt + delta, (PM, PMM, s, best, bt)
                worst = max(worst, best - bt)
        assert 0 < worst <= delta
    PM, PMM = 3, -2
    delta = min(PM, -PMM) - PMM
    vals = [(a, b) for a in range(0, PM + 1) for b in range(PMM, 1)]
    for n in range(1, 5):
        for table in itertools.product(vals, repeat=n):
            for pat in itertools.product((0, 1), repeat=n):
                s = [table[i][0] if pat[i] else table[i][1] for i in range(n)]
                best, bt = exact_best(s), pass1_bound(s)
                assert bt <= best <= bt + delta, (table, pat, best, bt)


def test_operand_encodings_are_exact():
    """the fp16 / e5m2 arithmetic of pass 1 is exact.  (1) every integer of magnitude <= 2048 is an fp16 value
    and sums of two such integers that stay within the range are exact (11-bit significand); (2) the five plane values of
    the 5/-4 scoring and 0 are e5m2 values = fp16 values whose low byte is zero, so the byte planes lose nothing; (3)
    non-negative fp16 bit patterns order like the values, so an integer max on the patterns is the max of the values."""
    import numpy as np
    ints = np.arange(-2048, 2049)
    assert (ints.astype(np.float16).astype(np.int64) == ints).all()
    a = np.arange(0, 2040, 7, dtype=np.int64)
    for b in (10, 1, -8, 5, -4, 0):
        assert ((a.astype(np.float16) + np.float16(b)).astype(np.int64) == a + b).all()
    for v in (10, 1, -8, 5, -4, 0):
        bits = int(np.array([v], dtype=np.float16).view(np.uint16)[0])
        assert bits & 0xFF == 0, v                                        # the high byte alone is the value
        assert float(np.array([bits & 0xFF00], dtype=np.uint16).view(np.float16)[0]) == v
    assert int(np.array([9], dtype=np.float16).view(np.uint16)[0]) & 0xFF != 0      # 9 (a 9/-7 scoring) is not an e5m2 value
    pos = np.arange(0, 2049).astype(np.float16).view(np.uint16).astype(np.int64)
    assert (np.diff(pos) > 0).all()
