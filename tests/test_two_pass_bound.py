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
