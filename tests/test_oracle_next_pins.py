"""Pins for the oracle's next-row functions: MaxSSmap_fast and base-quality
position-specific scoring.  As in test_oracle_pins.py none of them uses the function under test to
check itself: brute force over every scored sub-range written independently in Python (explicit sums), the
decimated-sequence reduction of MaxSSmap_fast to the already-pinned plain scan, the uniform-score reduction of the
PSSM functions to the already-pinned plain functions, closed-form phred values, exhaustive enumeration of fitting
alignments for the PSSM second stage, symmetry and scaling invariants.
"""
import os

import numpy as np
import pytest

import gen

from test_oracle_nw_pins import rle

MATCH, MISMATCH, GAP = 5, -4, -26
GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- independent brute force

def brute_top2_general(genome, F, V, read, pm, pmm, strands=3, step=1):
    """Every gap-free sub-range of the scored read positions (i = 0, step, 2*step, ...), explicit sums, no recurrence.
    pm/pmm: per-position match / mismatch scores of the read as given (forward)."""
    Gn, m = len(genome), len(read)
    nfrag = -(-Gn // F)
    veff = m - 1 if (V < 0 or V > m - 1) else V
    gp = list(genome) + [4] * (nfrag * F + m - Gn)
    cands = []
    for f in range(nfrag):
        end = f * F + F + veff
        entries = []
        for strand in (0, 1):
            if not strands & (1 << strand):
                continue
            if strand == 0:
                q, qm, qmm = list(read), list(pm), list(pmm)
            else:
                q = list(gen.revcomp(np.array(read, dtype=np.uint8)))
                qm, qmm = list(pm)[::-1], list(pmm)[::-1]
            for d in range(F):
                g = f * F + d
                pos = [i for i in range(0, m, step) if g + i < end]
                sc = [qm[i] if (q[i] < 4 and q[i] == gp[g + i]) else qmm[i] for i in pos]
                best = 0
                for a in range(len(sc)):
                    for b in range(a, len(sc)):
                        best = max(best, sum(sc[a:b + 1]))
                entries.append((-best, strand, d))
        negsc, strand, d = sorted(entries)[0]
        cands.append((negsc, f, d, strand))
    cands.sort()
    out = []
    for k in range(2):
        if k < len(cands):
            negsc, f, d, strand = cands[k]
            out.append([f, d, -negsc, strand])
        else:
            out.append([-1, 0, 0, 0])
    return np.array(out, dtype=np.int32)


def _tiny_case(rng):
    Gn = int(rng.integers(20, 61))
    genome = rng.integers(0, 4, size=Gn).astype(np.uint8)
    genome[rng.random(Gn) < 0.05] = 4
    m = int(rng.integers(1, 13))
    if rng.random() < 0.6 and Gn > m:
        p = int(rng.integers(0, Gn - m))
        read = genome[p:p + m].copy()
        flip = rng.random(m) < 0.2
        read[flip] = rng.integers(0, 5, size=int(flip.sum()))
    else:
        read = rng.integers(0, 5, size=m).astype(np.uint8)
    return genome, read, m


# ----------------------------------------------------------------------------- MaxSSmap_fast

@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("F", [1, 3, 7, 16])
def test_fast_against_bruteforce(oracle_mod, seed, F):
    rng = np.random.default_rng(7000 * F + seed)
    genome, read, m = _tiny_case(rng)
    for V in (0, 1, m - 1, -1):
        for strands in (1, 2, 3):
            want = brute_top2_general(genome, F, V, read, [MATCH] * m, [MISMATCH] * m, strands, step=2)
            got = oracle_mod.map_reads(genome, F, V, read[None, :], [m], strands=strands, fast=True)[0]
            assert got.tolist() == want.tolist(), (seed, F, V, strands, gen.decode(genome), gen.decode(read))


@pytest.mark.parametrize("seed", range(5))
def test_fast_is_plain_scan_of_decimated_sequences(oracle_mod, seed):
    """Window start g scores read positions 0,2,4,.. against genome positions g, g+2, g+4, ..: that is the plain
    (pinned) scan of R[0::2] at window start g//2 of the genome's parity class G[g%2::2].  With one fragment covering
    the genome and full look-ahead the best score of the fast scan is the max over both parity classes."""
    rng = np.random.default_rng(7100 + seed)
    Gn = int(rng.integers(300, 500))
    genome = rng.integers(0, 4, size=Gn).astype(np.uint8)
    m = int(rng.integers(20, 41))
    p = int(rng.integers(0, Gn - m))
    read = genome[p:p + m].copy()
    flip = rng.random(m) < 0.15
    read[flip] = (read[flip] + rng.integers(1, 4, size=int(flip.sum()))) % 4
    got = oracle_mod.map_reads(genome, Gn, -1, read[None, :], [m], strands=1, fast=True)[0, 0]
    rdec = read[0::2]
    per_class = []
    for par in (0, 1):
        gdec = genome[par::2]
        sc, dg = oracle_mod.fragment_scores(gdec, len(gdec), -1, rdec, strand=0)
        per_class.append((int(sc[0]), 2 * int(dg[0]) + par))
    best = max(s for s, _ in per_class)
    first_g = min(g for s, g in per_class if s == best)
    assert got.tolist() == [0, first_g, best, 0]
    # every window start on its own
    for g in rng.integers(0, Gn, size=20):
        g = int(g)
        one = oracle_mod.diagonal_score(genome[g % 2::2], Gn, -1, g // 2, rdec)
        # brute force on the window alone, explicit sums over the scored positions
        sub = [MATCH if (read[i] == genome[g + i]) else MISMATCH for i in range(0, m, 2) if g + i < Gn]
        b = 0
        for a in range(len(sub)):
            for e in range(a, len(sub)):
                b = max(b, sum(sub[a:e + 1]))
        assert one == b


def test_fast_closed_forms(oracle_mod):
    """An exact copy of a genome window scores ceil(m/2)*match (every scored position matches); scores stay within
    [0, ceil(m/2)*match]; a read whose even positions are all wrong but odd positions right scores like a non-match."""
    rng = np.random.default_rng(7200)
    genome = rng.integers(0, 4, size=3000).astype(np.uint8)
    for m in (1, 2, 7, 36, 100, 101):
        p = int(rng.integers(0, 3000 - m))
        read = genome[p:p + m].copy()
        out = oracle_mod.map_reads(genome, 250, -1, read[None, :], [m], strands=1, fast=True)[0]
        assert out[0, 2] == -(-m // 2) * MATCH
        if m >= 36:
            assert out[0, :2].tolist() == [p // 250, p % 250]
        assert 0 <= out[1, 2] <= -(-m // 2) * MATCH
        bad = read.copy()
        bad[0::2] = (bad[0::2] + 1) % 4          # only the scored positions are corrupted
        out_bad = oracle_mod.map_reads(genome, 250, -1, bad[None, :], [m], strands=1, fast=True)[0]
        plain_bad = oracle_mod.map_reads(genome, 250, -1, bad[None, :], [m], strands=1)[0]
        if m >= 36:
            assert out_bad[0, 2] < (m // 4) * MATCH             # the true locus is invisible to the fast scan
            assert plain_bad[0, 2] >= MATCH                     # while the plain scan still sees its odd positions


def test_fast_equals_pssm_with_zero_weight_on_odd_positions(oracle_mod):
    """Skipping a position and scoring it 0 either way give the same Kadane values (H and best unchanged by +0), so
    the fast scan equals the PSSM scan with (match, mismatch) at even and (0, 0) at odd positions -- on the forward
    strand, and on the reverse strand when m is odd (then reversed even positions stay even)."""
    rng = np.random.default_rng(7300)
    genome = rng.integers(0, 4, size=2000).astype(np.uint8)
    for m in (9, 33, 51):
        reads = np.stack([genome[p:p + m] for p in rng.integers(0, 2000 - m, size=6)])
        reads[3:] = gen.revcomp(reads[3:].reshape(-1)).reshape(3, m)[::-1]
        flip = rng.random(reads.shape) < 0.1
        reads[flip] = (reads[flip] + 1) % 4
        pm = np.zeros((6, m), dtype=np.int32); pmm = np.zeros((6, m), dtype=np.int32)
        pm[:, 0::2] = MATCH; pmm[:, 0::2] = MISMATCH
        a = oracle_mod.map_reads(genome, 128, -1, reads, [m] * 6, strands=3, fast=True)
        b = oracle_mod.oracle.map_reads_pssm(genome, 128, -1, reads, [m] * 6, pm, pmm, strands=3)
        assert a.tolist() == b.tolist()


# ----------------------------------------------------------------------------- phred -> PSSM

def test_phred_closed_forms(oracle_mod):
    """x = 1 - 10^(-Q/10): Q = 0, 10, 20, 30, 40 -> x = 0, .9, .99, .999, .9999; "match x x", "mismatch x x/3".
    With scale 30000 every product below is a whole number, so the expected values are exact."""
    gold = {}
    for line in open(os.path.join(GOLD, "pssm_phred.txt")):
        if line.startswith("#") or not line.strip():
            continue
        q, x, pm, pmm = line.split()
        gold[int(q)] = (float(x), int(pm), int(pmm))
    qs = np.array(sorted(gold), dtype=np.uint8)
    pm, pmm = oracle_mod.oracle.pssm_from_phred(qs, MATCH, MISMATCH, 30000)
    for q, a, b in zip(qs, pm, pmm):
        x, want_pm, want_pmm = gold[int(q)]
        assert a == want_pm == round(30000 * MATCH * x)
        assert b == want_pmm == round(30000 * MISMATCH * x / 3)
    # monotone in Q, bounded by the uniform scores, mismatch = -(4/15) match up to rounding
    allq = np.arange(0, 94, dtype=np.uint8)
    pm, pmm = oracle_mod.oracle.pssm_from_phred(allq, MATCH, MISMATCH, 16)
    assert (np.diff(pm) >= 0).all() and (np.diff(pmm) <= 0).all()
    assert pm[0] == 0 and pmm[0] == 0 and pm[-1] == 16 * MATCH and pmm[-1] == round(16 * MISMATCH / 3)
    assert (np.abs(pmm * 15 + pm * 4) <= 15 * 0.5 + 4 * 0.5 + 1e-9).all()


# ----------------------------------------------------------------------------- PSSM scan

@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("F", [1, 3, 7, 16])
def test_pssm_against_bruteforce(oracle_mod, seed, F):
    rng = np.random.default_rng(8000 * F + seed)
    genome, read, m = _tiny_case(rng)
    qual = rng.integers(0, 42, size=m).astype(np.uint8)
    pm, pmm = oracle_mod.oracle.pssm_from_phred(qual, MATCH, MISMATCH, 16)
    for V in (0, 1, m - 1, -1):
        for strands in (1, 2, 3):
            want = brute_top2_general(genome, F, V, read, pm, pmm, strands)
            got = oracle_mod.oracle.map_reads_pssm(genome, F, V, read[None, :], [m], pm[None, :], pmm[None, :], strands)[0]
            assert got.tolist() == want.tolist(), (seed, F, V, strands)


def test_pssm_uniform_reduces_to_plain_scan(oracle_mod):
    """pmatch = match, pmismatch = mismatch at every position is the paper's "trivial match or mismatch cost"
    (PAPER.md:41): records must equal the pinned plain scan's, ties included."""
    cfg = gen.config(1)
    genome, _ = cfg.genome()
    r = cfg.reads(genome)
    reads, lens = r["reads"][:12], r["lens"][:12]
    reads[6:] = np.stack([gen.revcomp(x) for x in reads[6:]])
    pm = np.full(reads.shape, MATCH, dtype=np.int32); pmm = np.full(reads.shape, MISMATCH, dtype=np.int32)
    a = oracle_mod.map_reads(genome, cfg.frag_len, -1, reads, lens, strands=3)
    b = oracle_mod.oracle.map_reads_pssm(genome, cfg.frag_len, -1, reads, lens, pm, pmm, strands=3)
    assert a.tolist() == b.tolist()
    # integer scaling of the table scales scores and moves nothing
    c = oracle_mod.oracle.map_reads_pssm(genome, cfg.frag_len, -1, reads, lens, 7 * pm, 7 * pmm, strands=3)
    assert (c[:, :, 2] == 7 * a[:, :, 2]).all() and (c[:, :, [0, 1, 3]] == a[:, :, [0, 1, 3]]).all()


def test_pssm_reverse_complement_symmetry(oracle_mod):
    """Mapping R with table t on the reverse strand = mapping revcomp(R) with the reversed table on the forward strand."""
    rng = np.random.default_rng(8100)
    genome = rng.integers(0, 4, size=4000).astype(np.uint8)
    m = 40
    reads = np.stack([genome[p:p + m] for p in rng.integers(0, 4000 - m, size=8)])
    flip = rng.random(reads.shape) < 0.1
    reads[flip] = (reads[flip] + 2) % 4
    qual = rng.integers(2, 42, size=reads.shape).astype(np.uint8)
    pm, pmm = oracle_mod.oracle.pssm_from_phred(qual, MATCH, MISMATCH, 16)
    rc = np.stack([gen.revcomp(x) for x in reads])
    a = oracle_mod.oracle.map_reads_pssm(genome, 200, -1, rc, [m] * 8, pm[:, ::-1].copy(), pmm[:, ::-1].copy(), strands=2)
    b = oracle_mod.oracle.map_reads_pssm(genome, 200, -1, reads, [m] * 8, pm, pmm, strands=1)
    assert (a[:, :, :3] == b[:, :, :3]).all()
    assert (a[:, 0, 3] == 1).all() and (b[:, 0, 3] == 0).all()


def test_pssm_exact_read_closed_form(oracle_mod):
    """An exact, unique copy of a genome window scores sum(pmatch) at its own window start; a low-quality position
    that is wrong costs less than a high-quality one (PAPER.md:61's point)."""
    rng = np.random.default_rng(8200)
    genome = rng.integers(0, 4, size=5000).astype(np.uint8)
    m, p = 60, 1234
    read = genome[p:p + m].copy()
    qual = rng.integers(5, 42, size=m).astype(np.uint8)
    pm, pmm = oracle_mod.oracle.pssm_from_phred(qual, MATCH, MISMATCH, 16)
    out = oracle_mod.oracle.map_reads_pssm(genome, 500, -1, read[None, :], [m], pm[None, :], pmm[None, :], strands=1)[0]
    assert out[0].tolist() == [p // 500, p % 500, int(pm.sum()), 0]
    lo, hi = int(np.argmin(qual[20:40])) + 20, int(np.argmax(qual[20:40])) + 20
    scores = []
    for pos in (lo, hi):
        bad = read.copy(); bad[pos] = (bad[pos] + 1) % 4
        o = oracle_mod.oracle.map_reads_pssm(genome, 500, -1, bad[None, :], [m], pm[None, :], pmm[None, :], strands=1)[0]
        assert o[0, :2].tolist() == [p // 500, p % 500]
        assert o[0, 2] == int(pm.sum()) - int(pm[pos]) + int(pmm[pos])      # whole read still one run (|pmm| small)
        scores.append(int(o[0, 2]))
    assert scores[0] >= scores[1]


# ----------------------------------------------------------------------------- PSSM second stage

def enumerate_fitting_pssm(q, w, pm, pmm, gap):
    m, L = len(q), len(w)
    out = []

    def rec(i, j, score, ops, j0):
        if i == m:
            out.append((score, j, j0, tuple(ops)))
        if i < m and j < L:
            s = pm[i] if (q[i] < 4 and q[i] == w[j]) else pmm[i]
            rec(i + 1, j + 1, score + s, ops + [0], j0)
        if i < m:
            rec(i + 1, j, score + gap, ops + [1], j0)
        if j < L and ops:
            rec(i, j + 1, score + gap, ops + [2], j0)

    for j0 in range(L + 1):
        rec(0, j0, 0, [], j0)
    return out


def _pick(alns):
    best = max(a[0] for a in alns)
    alns = [a for a in alns if a[0] == best]
    jend = min(a[1] for a in alns)
    alns = [a for a in alns if a[1] == jend]
    alns.sort(key=lambda a: tuple(reversed(a[3])))
    return alns[0]


@pytest.mark.parametrize("seed", range(30))
def test_nw_pssm_exhaustive_tiny(oracle_mod, seed):
    rng = np.random.default_rng(8300 + seed)
    m = int(rng.integers(1, 6))
    L = int(rng.integers(1, 8))
    w = rng.integers(0, 3, size=L).astype(np.uint8)
    q = rng.integers(0, 3, size=m).astype(np.uint8)
    qual = rng.integers(0, 30, size=m).astype(np.uint8)
    pm, pmm = oracle_mod.oracle.pssm_from_phred(qual, MATCH, MISMATCH, 4)
    gap = [-26 * 4, -12, -4, -20][seed % 4]
    strand = seed % 2
    score, jend, j0, ops = _pick(enumerate_fitting_pssm(q, w, pm, pmm, gap))
    hit = np.array([[[0, 0, 0, strand], [-1, 0, 0, 0]]], dtype=np.int32)
    # the oracle orients the read itself: hand it the read (and table) whose strand-oriented form is q
    rd = gen.revcomp(q) if strand else q
    tpm, tpmm = (pm[::-1].copy(), pmm[::-1].copy()) if strand else (pm, pmm)
    sc, pos, cig, nc = oracle_mod.oracle.nw_align_pssm(w, L, -1, rd[None, :], [m], hit, tpm[None, :], tpmm[None, :], gap,
                                                       pad=0, cigar_stride=2 * m + L + 2)
    assert int(sc[0]) == score
    assert int(pos[0]) == j0
    assert [int(x) for x in cig[0, :nc[0]]] == rle(ops)


def test_nw_pssm_uniform_reduces_to_plain_nw(oracle_mod):
    cfg = gen.config(1)
    genome, _ = cfg.genome()
    r = cfg.reads(genome)
    reads, lens = r["reads"][:10], r["lens"][:10]
    top2 = oracle_mod.map_reads(genome, cfg.frag_len, -1, reads, lens, strands=3)
    a = oracle_mod.nw_align(genome, cfg.frag_len, -1, reads, lens, top2)
    pm = np.full(reads.shape, MATCH, dtype=np.int32); pmm = np.full(reads.shape, MISMATCH, dtype=np.int32)
    b = oracle_mod.oracle.nw_align_pssm(genome, cfg.frag_len, -1, reads, lens, top2, pm, pmm, GAP)
    for x, y in zip(a, b):
        assert (x == y).all()


def test_both_builds_agree_on_next_rows(oracle_mod):
    cfg = gen.config(1)
    genome, _ = cfg.genome()
    r = cfg.reads(genome)
    reads, lens = r["reads"][:6], r["lens"][:6]
    rng = np.random.default_rng(8400)
    qual = rng.integers(2, 42, size=reads.shape).astype(np.uint8)
    pm2, pmm2 = oracle_mod.oracle.pssm_from_phred(qual, MATCH, MISMATCH, 16, opt="O2")
    pm3, pmm3 = oracle_mod.oracle.pssm_from_phred(qual, MATCH, MISMATCH, 16, opt="O3")
    assert (pm2 == pm3).all() and (pmm2 == pmm3).all()
    assert (oracle_mod.map_reads(genome, cfg.frag_len, 0, reads, lens, strands=3, fast=True, opt="O2")
            == oracle_mod.map_reads(genome, cfg.frag_len, 0, reads, lens, strands=3, fast=True, opt="O3")).all()
    assert (oracle_mod.oracle.map_reads_pssm(genome, cfg.frag_len, 0, reads, lens, pm2, pmm2, 3, opt="O2")
            == oracle_mod.oracle.map_reads_pssm(genome, cfg.frag_len, 0, reads, lens, pm2, pmm2, 3, opt="O3")).all()
