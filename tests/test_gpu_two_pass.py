"""-m gpu: the two-pass scan (scan variant 7).  Pass 1's fragment bounds are checked against the oracle's
exact per-fragment scores (u <= score <= u + delta for every read, strand and fragment), and the records of the two-pass
scan against the oracle, bit for bit, on the geometries where pruning can go wrong: ties, duplicated blocks, reads with
N, odd lengths, truncated look-ahead, ragged tiles, other scorings."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


def _cmp(got, want, ctx=""):
    bad = np.where((got != want).any(axis=(1, 2)))[0]
    assert bad.size == 0, f"{ctx}: {bad.size} reads differ, first {bad[0]}: got {got[bad[0]].tolist()} want {want[bad[0]].tolist()}"


def _bounds(G, reads, lens, strands, match=5, mismatch=-4, fast=False):
    import torch
    import paper_1403_2136_b200 as mss
    from gpu_util import to_dev
    rp, rn = gen.pack_reads(reads, lens)
    u, delta = mss.mss_map_reads_bounds(G, to_dev(rp), to_dev(rn), to_dev(np.asarray(lens, dtype=np.int32)),
                                        int(reads.shape[1]), mss.Scoring(match, mismatch, -26), strands, fast)
    torch.cuda.synchronize()
    return u.cpu().numpy().view(np.uint16).astype(np.int64), delta


def _exact_fragment_scores(oracle_mod, g, F, V, read, m, strand, match, mismatch, fast):
    if not fast:
        return oracle_mod.fragment_scores(g, F, V, read[:m], match=match, mismatch=mismatch, strand=strand, opt="O3")[0]
    # MaxSSmap_fast per fragment: the PSSM scan with zero weight on the skipped positions of the oriented query
    q = gen.revcomp(read[:m]) if strand else read[:m]
    pm = np.zeros(m, dtype=np.int32); pmm = np.zeros(m, dtype=np.int32)
    pm[0::2] = match; pmm[0::2] = mismatch
    nfrag = -(-g.size // F)
    out = np.zeros(nfrag, dtype=np.int64)
    # one fragment at a time through the pinned PSSM oracle on a genome cut to the fragment's readable window
    veff = m - 1 if (V < 0 or V > m - 1) else V
    for f in range(nfrag):
        sub = g[f * F: min(g.size, f * F + F + veff)]
        padn = np.full(F + veff, gen.N, dtype=np.uint8); padn[:sub.size] = sub
        r = oracle_mod.map_reads_pssm(padn, F, veff, q[None, :], [m], pm[None, :], pmm[None, :], strands=1)
        out[f] = r[0, 0, 2] if r[0, 0, 0] == 0 else (r[0, 1, 2] if r[0, 1, 0] == 0 else 0)
    return out


@pytest.mark.parametrize("F,V,m,match,mismatch,fast", [
    (1000, -1, 100, 5, -4, False), (1000, 0, 100, 5, -4, False), (4096, -1, 51, 5, -4, False), (700, 30, 77, 5, -4, False),
    (1000, -1, 100, 2, -7, False), (1000, -1, 101, 9, -3, False), (2048, -1, 36, 1, -1, False),
    (1000, -1, 100, 5, -4, True), (1000, 0, 51, 5, -4, True), (1000, -1, 75, 3, -5, True),
])
def test_pass1_bounds_hold(oracle_mod, F, V, m, match, mismatch, fast):
    from gpu_util import load_genome
    g = gen.make_genome(40_000, 31)[0]
    g[5000:5300] = gen.N
    r = gen.make_reads(g, 24, m, 3100 + m, sub_rate=0.15)
    reads, lens = r["reads"], r["lens"].copy()
    lens[5] = max(1, m - 7); reads[5, lens[5]:] = gen.N
    lens[9] = 1; reads[9, 1:] = gen.N
    G = load_genome(g, F, V)
    u, delta = _bounds(G, reads, lens, 3, match, mismatch, fast)
    assert delta == min(match, -mismatch) - mismatch
    for i in range(reads.shape[0]):
        for s in (0, 1):
            exact = _exact_fragment_scores(oracle_mod, g, F, V, reads[i], int(lens[i]), s, match, mismatch, fast)
            ui = u[i, s]
            assert (ui != 0xFFFF).all()
            assert (ui <= exact).all() and (exact <= ui + delta).all(), (i, s, int(np.argmax(np.abs(exact - ui))))


def test_pass1_marks_reads_with_n_as_unbounded(oracle_mod):
    from gpu_util import load_genome
    g = gen.make_genome(20_000, 32)[0]
    r = gen.make_reads(g, 6, 60, 3200, sub_rate=0.1)
    reads, lens = r["reads"].copy(), r["lens"]
    reads[2, 17] = gen.N
    G = load_genome(g, 1000, -1)
    u, _ = _bounds(G, reads, lens, 3)
    assert (u[2] == 0xFFFF).all() and (u[[0, 1, 3, 4, 5]] != 0xFFFF).all()


@pytest.mark.parametrize("strands", [1, 2, 3])
@pytest.mark.parametrize("F,V", [(1000, 0), (1000, -1), (1000, 17), (4096, -1), (700, 30), (300, -1), (5000, 50)])
def test_two_pass_records_equal_oracle(oracle_mod, F, V, strands):
    from gpu_util import load_genome, map_reads, map_reads_fast
    cfg = gen.config(1)
    g, _ = cfg.genome()
    r = cfg.reads(g)
    reads, lens = r["reads"][:64].copy(), r["lens"][:64].copy()
    reads[1::2] = np.stack([gen.revcomp(x) for x in reads[1::2]])
    reads[7, 40] = gen.N                                  # a read with an N takes the "every fragment" route
    lens[11] = 99; reads[11, 99:] = gen.N                 # odd length: the last double step has a single position
    G = load_genome(g, F, V)
    want = oracle_mod.map_reads_parallel(g, F, V, reads, lens, strands=strands)
    _cmp(map_reads(G, reads, lens, strands=strands, variant=7), want, f"two-pass F={F} V={V} strands={strands}")
    want = oracle_mod.map_reads_parallel(g, F, V, reads, lens, strands=strands, fast=True)
    _cmp(map_reads_fast(G, reads, lens, strands=strands, variant=7), want, f"two-pass fast F={F} V={V} strands={strands}")


def test_two_pass_ties_duplicates_and_zero_scores(oracle_mod):
    """Equal scores in several fragments (the pruning must keep every fragment that ties the second place), reads that
    match nowhere (all bounds 0: every fragment is a candidate) and a periodic genome."""
    from gpu_util import load_genome, map_reads
    rng = np.random.default_rng(3300)
    g = rng.integers(0, 4, size=24_000).astype(np.uint8)
    block = g[3 * 1000 + 100: 3 * 1000 + 400].copy()
    for f in (7, 12, 19):
        g[f * 1000 + 100: f * 1000 + 400] = block                   # four identical copies: fragments 3, 7, 12, 19
    reads = np.stack([block[50:150], block[100:200], gen.revcomp(block[20:120]),
                      np.full(100, 0, dtype=np.uint8), rng.integers(0, 4, size=100).astype(np.uint8)])
    lens = np.full(5, 100, dtype=np.int32)
    gz = g.copy(); gz[gz == 0] = 1                                   # no A in the genome: the all-A read scores 0 everywhere
    for genome in (g, gz):
        G = load_genome(genome, 1000, -1)
        want = oracle_mod.map_reads_parallel(genome, 1000, -1, reads, lens, strands=3)
        _cmp(map_reads(G, reads, lens, strands=3, variant=7), want, "ties")
    per = np.tile(np.array([0, 1], dtype=np.uint8), 6000)
    G = load_genome(per, 512, -1)
    rd = np.tile(np.array([0, 1], dtype=np.uint8), 30)[None, :]
    want = oracle_mod.map_reads_parallel(per, 512, -1, rd, [60], strands=3)
    _cmp(map_reads(G, rd, [60], strands=3, variant=7), want, "periodic")


def test_two_pass_other_scorings_and_long_reads(oracle_mod):
    from gpu_util import load_genome, map_reads
    g = gen.make_genome(30_000, 34)[0]
    r = gen.make_reads(g, 20, 90, 3400, sub_rate=0.2)
    G = load_genome(g, 1500, -1)
    for match, mismatch in ((1, -1), (2, -3), (9, -7), (10, -40), (3, -1)):
        want = oracle_mod.map_reads_parallel(g, 1500, -1, r["reads"], r["lens"], match=match, mismatch=mismatch, strands=3)
        _cmp(map_reads(G, r["reads"], r["lens"], match=match, mismatch=mismatch, variant=7), want, f"scoring {match}/{mismatch}")
    r = gen.make_reads(g, 6, 700, 3401, sub_rate=0.1)
    G = load_genome(g, 2048, -1)
    want = oracle_mod.map_reads_parallel(g, 2048, -1, r["reads"], r["lens"], strands=3)
    _cmp(map_reads(G, r["reads"], r["lens"], variant=7), want, "m=700")


def test_two_pass_chunk_loop(oracle_mod):
    """The bounds are produced per chunk of reads (1 GiB by default).  With a 20 kB limit the 200 reads of the tiny config
    take dozens of chunks (ragged last chunk included); the records must not change."""
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, map_reads
    cfg = gen.config(1)
    g, _ = cfg.genome()
    r = cfg.reads(g)
    reads, lens = r["reads"].copy(), r["lens"]
    reads[1::2] = np.stack([gen.revcomp(x) for x in reads[1::2]])
    want = oracle_mod.map_reads_parallel(g, cfg.frag_len, -1, reads, lens, strands=3)
    G = load_genome(g, cfg.frag_len, -1)
    try:
        for nbytes in (20_000, 1400, 200):                # 100, 7 and 1 reads per chunk (50 fragments x 2 strands x 2 B per read)
            mss.mss_set_two_pass_chunk_bytes(nbytes)
            got = map_reads(G, reads, lens, strands=3, variant=7)
            assert mss.mss_get_last_launch()["launches"] >= 2 * (200 * 200 // nbytes)
            _cmp(got, want, f"chunk bytes {nbytes}")
    finally:
        mss.mss_set_two_pass_chunk_bytes(0)
