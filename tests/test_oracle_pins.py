"""Pins for the CPU oracle's MaxSS stage (oracle/maxss_oracle.c) -- none of them calls the oracle to check
the oracle.  Each pin is something the paper or the mathematics fixes: the paper's Figure 2 toy, a brute
force over all gap-free substring pairs written independently in Python (explicit sums, sorted(), no
Kadane), closed forms, invariants and tie-break constructions (SURVEY.md section 8(c) "What pins each part").
"""
import os

import numpy as np
import pytest

import gen

GOLD = os.path.join(os.path.dirname(__file__), "golden")
MATCH, MISMATCH = 5, -4


# ----------------------------------------------------------------------------- independent brute force

def _s(a, b, match=MATCH, mismatch=MISMATCH):
    return match if (a == b and a < 4 and b < 4) else mismatch


def brute_top2(genome, F, V, read, strands=3, match=MATCH, mismatch=MISMATCH):
    """Enumerate every gap-free substring pair (read[a..b], genome[g+a..g+b]) -- no recurrence."""
    Gn = len(genome)
    nfrag = -(-Gn // F)
    m = len(read)
    veff = m - 1 if (V < 0 or V > m - 1) else V
    gp = list(genome) + [4] * (nfrag * F + m - Gn)
    cands = []
    for f in range(nfrag):
        end = f * F + F + veff
        entries = []
        for strand in (0, 1):
            if not strands & (1 << strand):
                continue
            q = list(read) if strand == 0 else list(gen.revcomp(np.array(read, dtype=np.uint8)))
            for d in range(F):
                g = f * F + d
                best = 0  # empty subsequence
                for a in range(m):
                    for b in range(a, m):
                        if g + b >= end:
                            break
                        tot = sum(_s(q[i], gp[g + i], match, mismatch) for i in range(a, b + 1))
                        best = max(best, tot)
                entries.append((-best, strand, d))
        negsc, strand, d = sorted(entries)[0]          # score desc, strand asc, diag asc
        cands.append((negsc, f, d, strand))
    cands.sort()                                       # score desc, fragment asc
    out = []
    for k in range(2):
        if k < len(cands):
            negsc, f, d, strand = cands[k]
            out.append([f, d, -negsc, strand])
        else:
            out.append([-1, 0, 0, 0])
    return np.array(out, dtype=np.int32)


# ----------------------------------------------------------------------------- the paper's own figures

def _gold(name):
    d = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        d[k] = v
    return d


def test_fig2_fragment_cutting(oracle_mod):
    """PAPER.md:273-281 Fig. 2: ACCGTAGGACCA, F=3 -> fragments ACC GTA GGA CCA (fragment f = [3f, 3f+3))."""
    gold = _gold("fig2_toy.txt")
    genome = gen.encode(gold["genome"][0])
    F = int(gold["frag_len"][0])
    frags = gold["fragments"]
    assert [gold["genome"][0][i:i + F] for i in range(0, len(genome), F)] == frags
    # the transposed matrix of the figure: column t holds fragment t (thread t reads A,G,G,C first)
    assert ["".join(fr[k] for fr in frags) for k in range(F)] == gold["transposed"]
    # each fragment, used as a read with no look-ahead, must come back as its own fragment at diagonal 0
    for f, fr in enumerate(frags):
        out = oracle_mod.map_reads(genome, F, 0, gen.encode(fr)[None, :], [F], strands=1)
        sc, dg = oracle_mod.fragment_scores(genome, F, 0, gen.encode(fr), strand=0)
        assert sc[f] == F * MATCH
        if fr != "ACC":       # "ACC" also occurs at genome position 8 = fragment 2, diag 2, read into fragment 3: not with V=0
            assert out[0, 0].tolist() == [f, 0, F * MATCH, 0]
    # a read across the junction of fragments 0|1: CGT starts at genome position 2 = fragment 0, diagonal 2
    out = oracle_mod.map_reads(genome, F, -1, gen.encode("CGT")[None, :], [3], strands=1)
    assert out[0, 0].tolist() == [0, 2, 15, 0]
    # without look-ahead the window start at 2 sees only 'C' (score 5).  By hand, per fragment:
    # ACC: d=1 lays C on C (5); GTA: no window start lays any read base on an equal base (0);
    # GGA: d=0 lays read G on the second G (5); CCA: d=0 lays C on C (5).
    sc, dg = oracle_mod.fragment_scores(genome, F, 0, gen.encode("CGT"), strand=0)
    assert sc.tolist() == [5, 0, 5, 5] and dg.tolist() == [1, 0, 0, 0]


def test_thread_counts_of_the_paper():
    """5 Mbp / 4800 -> 1042 threads, /48000 -> 104, /480000 -> 11 (nfrag arithmetic)."""
    gold = _gold("paper_constants.txt")
    G = int(gold["genome_bp"][0])
    for F, want in zip(map(int, gold["frag_lens"]), map(int, gold["threads"])):
        nfrag = -(-G // F)
        # the paper rounds ("about 1042", "104" for 104.17): ceil or floor must hit the printed value
        assert want in (nfrag, G // F), (F, nfrag)


def test_padding_rule(oracle_mod):
    """last fragment padded with N; nfrag = ceil(G/F); padded positions score as mismatches."""
    genome = gen.encode("ACGTACGTAC")            # G = 10, F = 4 -> 3 fragments, last = AC NN
    sc, dg = oracle_mod.fragment_scores(genome, 4, -1, gen.encode("ACGT"), strand=0)
    assert len(sc) == 3
    assert sc.tolist() == [20, 20, 10] and dg.tolist() == [0, 0, 0]


# ----------------------------------------------------------------------------- brute force

@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("F", [1, 3, 7, 16])
def test_against_bruteforce(oracle_mod, seed, F):
    rng = np.random.default_rng(1000 * F + seed)
    Gn = int(rng.integers(20, 61))
    genome = rng.integers(0, 4, size=Gn).astype(np.uint8)
    genome[rng.random(Gn) < 0.05] = 4
    m = int(rng.integers(1, 13))
    # half of the reads are (noisy) copies of a genome window so that high scores and ties occur
    if rng.random() < 0.5 and Gn > m:
        p = int(rng.integers(0, Gn - m))
        read = genome[p:p + m].copy()
        flip = rng.random(m) < 0.2
        read[flip] = rng.integers(0, 5, size=int(flip.sum()))
    else:
        read = rng.integers(0, 5, size=m).astype(np.uint8)
    for V in (0, 1, m - 1, -1, m + 5):
        for strands in (1, 2, 3):
            want = brute_top2(genome, F, V, read, strands)
            got = oracle_mod.map_reads(genome, F, V, read[None, :], [m], strands=strands)[0]
            assert got.tolist() == want.tolist(), (seed, F, V, strands, gen.decode(genome), gen.decode(read))


def test_bruteforce_other_scores(oracle_mod):
    rng = np.random.default_rng(7)
    genome = rng.integers(0, 4, size=40).astype(np.uint8)
    read = genome[10:19].copy()
    read[4] = (read[4] + 1) % 4
    for match, mismatch in ((1, -1), (2, -3), (7, -1)):
        want = brute_top2(genome, 8, -1, read, 3, match, mismatch)
        got = oracle_mod.map_reads(genome, 8, -1, read[None, :], [9], match=match, mismatch=mismatch, strands=3)[0]
        assert got.tolist() == want.tolist()


# ----------------------------------------------------------------------------- closed forms

def _tiny():
    cfg = gen.config(1)
    g, _ = cfg.genome()
    return cfg, g


def _unique(genome, sub):
    gb, sb = genome.tobytes(), sub.tobytes()
    first = gb.find(sb)
    return first >= 0 and gb.find(sb, first + 1) < 0


def test_exact_read_scores_m_times_match(oracle_mod):
    cfg, g = _tiny()
    rng = np.random.default_rng(3)
    F = 1000
    for m in (1, 17, 100, 250):
        for _ in range(3):
            p = int(rng.integers(0, g.size - m))
            read = g[p:p + m].copy()
            out = oracle_mod.map_reads(g, F, -1, read[None, :], [m], strands=1)[0]
            assert out[0, 2] == m * MATCH
            if m >= 17:
                assert _unique(g, read)
                assert out[0].tolist() == [p // F, p % F, m * MATCH, 0]
                assert out[1, 2] < m * MATCH


def test_score_range_and_all_n(oracle_mod):
    cfg, g = _tiny()
    r = cfg.reads(g)
    out = oracle_mod.map_reads(g, 1000, 0, r["reads"][:20], r["lens"][:20], strands=3)
    assert (out[:, :, 2] >= 0).all() and (out[:, :, 2] <= 100 * MATCH).all()
    alln = np.full((1, 30), 4, dtype=np.uint8)
    got = oracle_mod.map_reads(g[:5000], 1000, -1, alln, [30], strands=3)[0]
    # a fragment scoring 0 is still a fragment: best = fragment 0, second = fragment 1, diag 0, forward
    assert got.tolist() == [[0, 0, 0, 0], [1, 0, 0, 0]]
    gn = np.full(3000, 4, dtype=np.uint8)
    got = oracle_mod.map_reads(gn, 1000, -1, g[None, :50], [50], strands=3)[0]
    assert got.tolist() == [[0, 0, 0, 0], [1, 0, 0, 0]]
    # one fragment only: no second fragment
    got = oracle_mod.map_reads(g[:700], 1000, -1, g[None, 100:150], [50], strands=1)[0]
    assert got.tolist() == [[0, 100, 250, 0], [-1, 0, 0, 0]]


def _max_subarray(x):
    """max over a<=b of sum(x[a..b]), >= 0, from prefix sums (not Kadane)."""
    pre = np.concatenate([[0], np.cumsum(x)])
    best = 0
    for a in range(len(x)):
        best = max(best, int((pre[a + 1:] - pre[a]).max()))
    return best


def test_known_substitution_pattern(oracle_mod):
    cfg, g = _tiny()
    rng = np.random.default_rng(11)
    F = 1000
    for _ in range(5):
        m = 100
        p = int(rng.integers(0, g.size - m))
        pat = rng.random(m) < 0.15
        read = g[p:p + m].copy()
        read[pat] = (read[pat] + rng.integers(1, 4, size=int(pat.sum()))) % 4
        want = _max_subarray(np.where(pat, MISMATCH, MATCH))
        assert oracle_mod.diagonal_score(g, F, -1, p, read) == want
        out = oracle_mod.map_reads(g, F, -1, read[None, :], [m], strands=3)[0]
        assert out[0, 2] >= want
        if want > 200:  # far above the random background (~80): the true diagonal wins
            assert out[0].tolist()[:2] == [p // F, p % F] and out[0, 3] == 0


def test_truncation_closed_form(oracle_mod):
    """V = 0: only the in-fragment prefix of the read counts: match * (F - p mod F)."""
    cfg, g = _tiny()
    F, m = 1000, 100
    for p in (950, 2999, 7901, 13990):
        read = g[p:p + m].copy()
        assert p % F > F - m
        assert oracle_mod.diagonal_score(g, F, 0, p, read) == MATCH * (F - p % F)
        assert oracle_mod.diagonal_score(g, F, 10, p, read) == MATCH * min(m, F - p % F + 10)
        assert oracle_mod.diagonal_score(g, F, -1, p, read) == MATCH * m
        assert oracle_mod.diagonal_score(g, F, 10_000, p, read) == MATCH * m


# ----------------------------------------------------------------------------- invariants

def test_reverse_complement_symmetry(oracle_mod):
    cfg, g = _tiny()
    r = gen.make_reads(g, 12, 60, 99, sub_rate=0.15, both_strands=True)
    reads, lens = r["reads"], r["lens"]
    rc = gen.revcomp(reads)
    a = oracle_mod.map_reads(g, 1000, -1, reads, lens, strands=2)
    b = oracle_mod.map_reads(g, 1000, -1, rc, lens, strands=1)
    assert (a[:, :, :3] == b[:, :, :3]).all()
    assert (a[:, :, 3] == 1).all() and (b[:, :, 3] == 0).all()
    both = oracle_mod.map_reads(g, 1000, -1, reads, lens, strands=3)
    f = oracle_mod.map_reads(g, 1000, -1, reads, lens, strands=1)
    assert (both[:, 0, 2] == np.maximum(a[:, 0, 2], f[:, 0, 2])).all()
    # planted reads come back on the strand they were drawn from
    planted = both[:, 0, 2] > 130
    assert planted.sum() >= 5 and (both[planted, 0, 3] == r["strand"][planted]).all()


def test_whole_genome_equals_max_over_fragments(oracle_mod):
    """With look-ahead m-1 the best score and its lowest global diagonal do not depend on F."""
    g = gen.make_genome(6000, 5)[0]
    r = gen.make_reads(g, 6, 40, 6, sub_rate=0.2, both_strands=False)
    ref = None
    for F in (6000, 7000, 4096, 1000, 37, 1):
        for strand in (0, 1):
            rows = []
            for k in range(6):
                sc, dg = oracle_mod.fragment_scores(g, F, -1, r["reads"][k], strand=strand)
                f = int(np.argmax(sc))                      # first maximiser = lowest fragment
                rows.append((int(sc[f]), f * F + int(dg[f])))
            if F == 6000:
                ref = ref or {}
                ref[strand] = rows
            assert rows == ref[strand], (F, strand)


def test_monotone_scaling_and_n_padding(oracle_mod):
    cfg, g = _tiny()
    r = cfg.reads(g)
    reads, lens = r["reads"][:10], r["lens"][:10]
    for k in range(10):
        s0, _ = oracle_mod.fragment_scores(g, 1000, 0, reads[k])
        s1, _ = oracle_mod.fragment_scores(g, 1000, 30, reads[k])
        s2, _ = oracle_mod.fragment_scores(g, 1000, -1, reads[k])
        assert (s0 <= s1).all() and (s1 <= s2).all()
    a = oracle_mod.map_reads(g, 1000, -1, reads, lens, strands=3)
    b = oracle_mod.map_reads(g, 1000, -1, reads, lens, match=15, mismatch=-12, strands=3)
    assert (b[:, :, 2] == 3 * a[:, :, 2]).all() and (b[:, :, [0, 1, 3]] == a[:, :, [0, 1, 3]]).all()
    padded = np.concatenate([reads, np.full((10, 7), 4, dtype=np.uint8)], axis=1)
    c = oracle_mod.map_reads(g, 1000, -1, padded, lens + 7, strands=1)
    d = oracle_mod.map_reads(g, 1000, -1, reads, lens, strands=1)
    assert (c == d).all()
    # bytes beyond lens[r] are ignored
    junk = padded.copy()
    junk[:, 100:] = 2
    e = oracle_mod.map_reads(g, 1000, -1, junk, lens, strands=1)
    assert (e == d).all()


# ----------------------------------------------------------------------------- tie-breaks

def test_ties_lowest_fragment(oracle_mod):
    rng = np.random.default_rng(21)
    F = 100
    g = rng.integers(0, 4, size=1000).astype(np.uint8)
    block = rng.integers(0, 4, size=60).astype(np.uint8)
    g[320:380] = block
    g[725:785] = block
    out = oracle_mod.map_reads(g, F, -1, block[None, :], [60], strands=1)[0]
    assert out.tolist() == [[3, 20, 300, 0], [7, 25, 300, 0]]


def test_ties_forward_strand_and_lowest_diag(oracle_mod):
    pal = gen.encode("ACGTTGCAACGT" + "ACGTTGCAACGT")      # its own reverse complement
    assert (gen.revcomp(pal) == pal).all()
    rng = np.random.default_rng(22)
    g = rng.integers(0, 4, size=600).astype(np.uint8)
    g[250:274] = pal
    out = oracle_mod.map_reads(g, 100, -1, pal[None, :], [24], strands=3)[0]
    assert out[0].tolist() == [2, 50, 120, 0]
    periodic = gen.encode("AC" * 100)
    read = gen.encode("ACACACAC")
    out = oracle_mod.map_reads(periodic, 50, -1, read[None, :], [8], strands=1)[0]
    assert out.tolist() == [[0, 0, 40, 0], [1, 0, 40, 0]]


def test_second_is_a_distinct_fragment(oracle_mod):
    """The same fragment on the other strand, or at another diagonal, is not a second place (reading 8)."""
    rng = np.random.default_rng(23)
    g = rng.integers(0, 4, size=400).astype(np.uint8)
    read = g[110:150].copy()
    g[160:200] = read                      # second copy in the same fragment (F = 100)
    out = oracle_mod.map_reads(g, 100, -1, read[None, :], [40], strands=3)[0]
    assert out[0].tolist() == [1, 10, 200, 0]
    assert out[1, 0] != 1 and out[1, 2] < 200


# ----------------------------------------------------------------------------- builds agree; fan-out agrees

def test_o2_o3_and_parallel_agree(oracle_mod):
    cfg, g = _tiny()
    r = cfg.reads(g)
    a = oracle_mod.map_reads(g, cfg.frag_len, cfg.overlap, r["reads"][:24], r["lens"][:24], strands=3, opt="O2")
    b = oracle_mod.map_reads(g, cfg.frag_len, cfg.overlap, r["reads"][:24], r["lens"][:24], strands=3, opt="O3")
    c = oracle_mod.map_reads_parallel(g, cfg.frag_len, cfg.overlap, r["reads"][:24], r["lens"][:24], strands=3,
                                      workers=3)
    assert (a == b).all() and (a == c).all()
    # the generator's truth: the planted fragment wins for (almost) every Tiny read (context)
    assert (np.abs(a[:, 0, 0] - r["start"][:24] // 1000) <= 1).mean() > 0.9
