"""Pins for the oracle's second stage (oracle_nw_align): exhaustive enumeration of every fitting alignment on
tiny inputs (no DP), closed forms, re-scoring of the CIGAR, planted single indels, hand-made tie cases.
Readings 14-16 of DESIGN.md section 3 (fitting alignment, linear gap, smallest end column, M > I > D)."""
import numpy as np
import pytest

import gen

MATCH, MISMATCH, GAP = 5, -4, -26


def _s(a, b, match=MATCH, mismatch=MISMATCH):
    return match if (a == b and a < 4 and b < 4) else mismatch


def enumerate_fitting(q, w, match=MATCH, mismatch=MISMATCH, gap=GAP):
    """All alignments of the whole of q to a substring of w: (score, end_col, start_col, ops in read order).

    ops: 0 = M (read base on window base), 1 = I (read base on nothing), 2 = D (window base skipped).
    A leading D is not an alignment of the read (row 0 of the recurrence is free), so paths start with M or I."""
    m, L = len(q), len(w)
    out = []

    def rec(i, j, score, ops, j0):
        if i == m:
            out.append((score, j, j0, tuple(ops)))
        if i < m and j < L:
            rec(i + 1, j + 1, score + _s(q[i], w[j], match, mismatch), ops + [0], j0)
        if i < m:
            rec(i + 1, j, score + gap, ops + [1], j0)
        if j < L and ops:       # trailing D's are legal cells of the recurrence (never optimal, kept for completeness)
            rec(i, j + 1, score + gap, ops + [2], j0)

    for j0 in range(L + 1):
        rec(0, j0, 0, [], j0)
    return out


def pick(alns):
    """max score; smallest end column; then, walking the ops from the END, prefer M over I over D."""
    best = max(a[0] for a in alns)
    alns = [a for a in alns if a[0] == best]
    jend = min(a[1] for a in alns)
    alns = [a for a in alns if a[1] == jend]
    alns.sort(key=lambda a: tuple(reversed(a[3])))
    return alns[0]


def rle(ops):
    out = []
    for op in ops:
        if out and out[-1][1] == op:
            out[-1][0] += 1
        else:
            out.append([1, op])
    return [(n << 4) | op for n, op in out]


def run_oracle(oracle_mod, window, q, pad=0, **kw):
    """Align q to the whole of `window` = a one-fragment genome with pad 0 and full look-ahead."""
    hit = np.array([[[0, 0, 0, 0], [-1, 0, 0, 0]]], dtype=np.int32)
    sc, pos, cig, nc = oracle_mod.nw_align(window, len(window), -1, np.asarray(q, dtype=np.uint8)[None, :], [len(q)],
                                           hit, pad=pad, cigar_stride=2 * len(q) + len(window) + 2, **kw)
    return int(sc[0]), int(pos[0]), [int(x) for x in cig[0, :nc[0]]]


@pytest.mark.parametrize("seed", range(40))
def test_exhaustive_tiny(oracle_mod, seed):
    rng = np.random.default_rng(500 + seed)
    m = int(rng.integers(1, 6))
    L = int(rng.integers(1, 8))
    w = rng.integers(0, 3, size=L).astype(np.uint8)       # small alphabet -> many ties
    q = rng.integers(0, 3, size=m).astype(np.uint8)
    gap = [-26, -3, -1, -5][seed % 4]                      # cheap gaps make I/D appear in optimal paths
    score, jend, j0, ops = pick(enumerate_fitting(q, w, gap=gap))
    got = run_oracle(oracle_mod, w, q, gap=gap)
    assert got[0] == score
    assert got[1] == j0
    assert got[2] == rle(ops), (gen.decode(w), gen.decode(q), gap)


def rescore(window_codes, ws, q, pos, cigar, match=MATCH, mismatch=MISMATCH, gap=GAP):
    i, j, tot = 0, pos - ws, 0
    for c in cigar:
        n, op = c >> 4, c & 15
        for _ in range(n):
            if op == 0:
                tot += _s(q[i], window_codes[j], match, mismatch); i += 1; j += 1
            elif op == 1:
                tot += gap; i += 1
            else:
                tot += gap; j += 1
    return tot, i


def test_exact_substring_and_hamming(oracle_mod):
    g = gen.make_genome(3000, 77)[0]
    q = g[1234:1234 + 80].copy()
    hit = np.array([[[1, 234, 400, 0], [-1, 0, 0, 0]]], dtype=np.int32)
    sc, pos, cig, nc = oracle_mod.nw_align(g, 1000, -1, q[None, :], [80], hit)
    assert sc[0] == 400 and pos[0] == 1234 and nc[0] == 1 and cig[0, 0] == (80 << 4)
    # window exactly as long as the read and prohibitive gaps -> the full-diagonal (Hamming-style) sum
    rng = np.random.default_rng(5)
    w = rng.integers(0, 4, size=50).astype(np.uint8)
    q = w.copy()
    mut = rng.random(50) < 0.3
    q[mut] = (q[mut] + 1) % 4
    want = int(np.where(mut, MISMATCH, MATCH).sum())
    got = run_oracle(oracle_mod, w, q, gap=-10**6)
    assert got == (want, 0, [50 << 4])


def test_reverse_strand_hit(oracle_mod):
    g = gen.make_genome(3000, 78)[0]
    q = gen.revcomp(g[2100:2160])
    hit = np.array([[[2, 100, 300, 1], [-1, 0, 0, 0]]], dtype=np.int32)
    sc, pos, cig, nc = oracle_mod.nw_align(g, 1000, -1, q[None, :], [60], hit)
    assert sc[0] == 300 and pos[0] == 2100 and cig[0, 0] == (60 << 4) and nc[0] == 1


@pytest.mark.parametrize("k", [1, 7, 30])
def test_planted_single_indel(oracle_mod, k):
    """aM kD bM / aM kI bM for an otherwise exact read with long flanks (26k < what a flank would lose un-gapped)."""
    g = gen.make_genome(4000, 79)[0]
    a, b = 200, 210
    p = 1500
    # deletion from the read (genome bases skipped): read = g[p:p+a] + g[p+a+k : p+a+k+b]
    q = np.concatenate([g[p:p + a], g[p + a + k:p + a + k + b]])
    hit = np.array([[[1, 0, 0, 0], [-1, 0, 0, 0]]], dtype=np.int32)
    sc, pos, cig, nc = oracle_mod.nw_align(g, 1000, -1, q[None, :], [a + b], hit)
    assert 26 * k < 6 * min(a, b)      # an un-gapped flank loses ~6.75 per base on random sequence
    assert pos[0] == p and sc[0] == 5 * (a + b) - 26 * k
    ops = [(int(c) >> 4, int(c) & 15) for c in cig[0, :nc[0]]]
    # with a linear gap cost the k skipped bases may slide over / split around equal flanking bases at no cost, so
    # the op *content* is pinned (k D's, a+b M's, no I, M at both ends) and re-scoring pins where they sit
    assert sum(n for n, o in ops if o == 2) == k and sum(n for n, o in ops if o == 0) == a + b
    assert all(o != 1 for _, o in ops) and ops[0][1] == 0 and ops[-1][1] == 0
    if k == 1:
        assert [o for _, o in ops] == [0, 2, 0]
    tot, used = rescore(g, 0, q, int(pos[0]), [int(c) for c in cig[0, :nc[0]]])
    assert tot == sc[0] and used == a + b
    # insertion into the read
    rng = np.random.default_rng(k)
    ins = rng.integers(0, 4, size=k).astype(np.uint8)
    q = np.concatenate([g[p:p + a], ins, g[p + a:p + a + b]])
    sc, pos, cig, nc = oracle_mod.nw_align(g, 1000, -1, q[None, :], [a + k + b], hit)
    ops = [(int(c) >> 4, int(c) & 15) for c in cig[0, :nc[0]]]
    assert pos[0] == p and sc[0] >= 5 * (a + b) - 26 * k
    if sc[0] == 5 * (a + b) - 26 * k:
        assert sum(n for n, o in ops if o == 1) == k and all(o != 2 for _, o in ops)
    tot, used = rescore(g, 0, q, int(pos[0]), [int(c) for c in cig[0, :nc[0]]])
    assert tot == sc[0] and used == a + k + b


def test_cigar_rescoring_and_bounds_on_tiny_config(oracle_mod):
    cfg = gen.config(1)
    g, _ = cfg.genome()
    r = cfg.reads(g)
    reads, lens = r["reads"][:60], r["lens"][:60]
    top2 = oracle_mod.map_reads(g, cfg.frag_len, cfg.overlap, reads, lens, strands=3)
    sc, pos, cig, nc = oracle_mod.nw_align(g, cfg.frag_len, cfg.overlap, reads, lens, top2)
    for k in range(60):
        q = reads[k] if top2[k, 0, 3] == 0 else gen.revcomp(reads[k])
        tot, used = rescore(g, 0, q, int(pos[k]), [int(c) for c in cig[k, :nc[k]]])
        assert tot == sc[k] and used == lens[k]
        assert sc[k] <= MATCH * lens[k]
        # lower bound: the best *full* (un-clamped) diagonal sum inside the window
        f = int(top2[k, 0, 0])
        ws, we = max(0, f * 1000 - 30), min(g.size, f * 1000 + 1000 + 0 + 30)
        full = max(sum(_s(q[i], g[j + i]) for i in range(100)) for j in range(ws, we - 100 + 1))
        assert sc[k] >= full
        # NW (gaps allowed, both flanks charged) vs MaxSS (best clamped run): NW >= MaxSS run minus the rest as mismatches
        assert sc[k] >= top2[k, 0, 2] - 4 * 100


def test_no_hit_and_window_clipping(oracle_mod):
    g = gen.make_genome(500, 80)[0]
    q = g[0:40].copy()
    hit = np.array([[[-1, 0, 0, 0], [-1, 0, 0, 0]]], dtype=np.int32)
    sc, pos, cig, nc = oracle_mod.nw_align(g, 100, -1, q[None, :], [40], hit)
    assert (sc[0], pos[0], nc[0]) == (0, -1, 0)
    # window clipped at the genome start and end
    hit = np.array([[[0, 0, 200, 0], [-1, 0, 0, 0]]], dtype=np.int32)
    sc, pos, cig, nc = oracle_mod.nw_align(g, 100, -1, q[None, :], [40], hit)
    assert (sc[0], pos[0]) == (200, 0)
    q = g[470:500].copy()
    hit = np.array([[[4, 70, 150, 0], [-1, 0, 0, 0]]], dtype=np.int32)
    sc, pos, cig, nc = oracle_mod.nw_align(g, 100, -1, q[None, :], [30], hit)
    assert (sc[0], pos[0]) == (150, 470)
    # read longer than the window: the overhang must be inserted (I), pinned by enumeration
    w = gen.encode("ACG")
    qq = gen.encode("TACGT")
    score, jend, j0, ops = pick(enumerate_fitting(qq, w, gap=-2))
    got = run_oracle(oracle_mod, w, qq, gap=-2)
    assert got == (score, j0, rle(ops))


def test_tie_order_hand_cases(oracle_mod):
    # q = AA, w = AAA: three diagonals score 10; smallest end column 2 -> start 0
    assert run_oracle(oracle_mod, gen.encode("AAA"), gen.encode("AA")) == (10, 0, [2 << 4])
    # q = AC vs w = AGC with gap -1: A-C aligned as M D M (5-1+5 = 9) beats MM (5-4 = 1)
    assert run_oracle(oracle_mod, gen.encode("AGC"), gen.encode("AC"), gap=-1) == (9, 0, [(1 << 4), (1 << 4) | 2, (1 << 4)])
    # q = AGC vs w = AC with gap -1: M I M
    assert run_oracle(oracle_mod, gen.encode("AC"), gen.encode("AGC"), gap=-1) == (9, 0, [(1 << 4), (1 << 4) | 1, (1 << 4)])
    # tie between M-then-gap and gap-then-M: q = AA, w = A, gap -4 = mismatch... (m=2, L=1): paths MI (5-4), IM (-4+5): end col 1 both;
    # walking back from the end: last op M (path IM) preferred over last op I (path MI)
    assert run_oracle(oracle_mod, gen.encode("A"), gen.encode("AA"), gap=-4) == (1, 0, [(1 << 4) | 1, (1 << 4)])
