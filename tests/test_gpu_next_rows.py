"""-m gpu: the next rows through the C ABI against the CPU oracle, bit-exact:
MaxSSmap_fast, base-quality position-specific scoring in both phases."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tiny():
    cfg = gen.config(1)
    g, _ = cfg.genome()
    r = cfg.reads(g)
    # half of the reads reverse-complemented so that both strands carry true hits
    reads = r["reads"].copy()
    reads[1::2] = np.stack([gen.revcomp(x) for x in reads[1::2]])
    quals = gen.make_quals(reads.shape[0], reads.shape[1], gen.S0 + 19)
    return cfg, g, reads, r["lens"], quals


def _cmp(got, want, ctx=""):
    bad = np.where((got != want).any(axis=(1, 2)))[0]
    assert bad.size == 0, f"{ctx}: {bad.size} reads differ, first {bad[0]}: got {got[bad[0]].tolist()} want {want[bad[0]].tolist()}"


# ----------------------------------------------------------------------------- MaxSSmap_fast

@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5, 6, 7])
def test_fast_tiny_every_variant(oracle_mod, tiny, variant):
    from gpu_util import load_genome, map_reads_fast
    cfg, g, reads, lens, _ = tiny
    want = oracle_mod.map_reads_parallel(g, cfg.frag_len, -1, reads, lens, strands=3, fast=True)
    G = load_genome(g, cfg.frag_len, -1)
    got = map_reads_fast(G, reads, lens, strands=3, variant=variant)
    _cmp(got, want, f"fast variant {variant}")


@pytest.mark.parametrize("strands", [1, 2, 3])
@pytest.mark.parametrize("F,V", [(1000, 0), (1000, 17), (4096, -1), (300, -1), (50_000, -1), (100, -1)])
def test_fast_geometries(oracle_mod, tiny, F, V, strands):
    from gpu_util import load_genome, map_reads_fast
    cfg, g, reads, lens, _ = tiny
    want = oracle_mod.map_reads_parallel(g, F, V, reads[:40], lens[:40], strands=strands, fast=True)
    G = load_genome(g, F, V)
    got = map_reads_fast(G, reads[:40], lens[:40], strands=strands)
    _cmp(got, want, f"fast F={F} V={V} strands={strands}")


def test_fast_mixed_and_odd_lengths(oracle_mod, tiny):
    """Ragged batch: lengths 1..101, odd and even (on the reverse strand the scored positions are those of the
    reverse-complemented read, so odd/even lengths differ), N bases in reads."""
    from gpu_util import load_genome, map_reads_fast
    cfg, g, _, _, _ = tiny
    rng = np.random.default_rng(4242)
    n, M = 48, 101
    lens = rng.integers(1, M + 1, size=n).astype(np.int32)
    lens[:4] = [1, 2, 3, M]
    reads = np.full((n, M), gen.N, dtype=np.uint8)
    for i in range(n):
        p = int(rng.integers(0, g.size - M))
        rd = g[p:p + lens[i]].copy()
        flip = rng.random(lens[i]) < 0.1
        rd[flip] = rng.integers(0, 5, size=int(flip.sum()))
        reads[i, :lens[i]] = gen.revcomp(rd) if i % 2 else rd
    want = oracle_mod.map_reads_parallel(g, 1000, -1, reads, lens, strands=3, fast=True)
    G = load_genome(g, 1000, -1)
    _cmp(map_reads_fast(G, reads, lens, strands=3), want, "fast ragged")


# ----------------------------------------------------------------------------- PSSM

def test_pssm_build_matches_oracle_table(oracle_mod, tiny):
    """Every phred value 0..93 (and values above, clamped to 93) against the oracle's double-precision table."""
    from gpu_util import pssm_tables
    q = np.arange(0, 120, dtype=np.uint8)[None, :].repeat(3, axis=0)
    lens = np.array([120, 60, 1], dtype=np.int32)
    for scale, match, mismatch in [(16, 5, -4), (1, 5, -4), (100, 5, -4), (7, 3, -11)]:
        _, pm, pmm = pssm_tables(q, lens, match, mismatch, scale)
        wpm, wpmm = oracle_mod.pssm_from_phred(np.minimum(q, 93), match, mismatch, scale)
        for r in range(3):
            assert (pm[r, :lens[r]] == wpm[r, :lens[r]]).all() and (pmm[r, :lens[r]] == wpmm[r, :lens[r]]).all()
            assert (pm[r, lens[r]:] == 0).all() and (pmm[r, lens[r]:] == 0).all()


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5, 6, 7])
def test_pssm_tiny_every_variant(oracle_mod, tiny, variant):
    from gpu_util import load_genome, map_reads_pssm, pssm_tables
    cfg, g, reads, lens, quals = tiny
    d_pssm, pm, pmm = pssm_tables(quals, lens)
    wpm, wpmm = oracle_mod.pssm_from_phred(quals, 5, -4, 16)
    assert (pm == wpm).all() and (pmm == wpmm).all()
    want = oracle_mod.map_reads_pssm_parallel(g, cfg.frag_len, -1, reads, lens, wpm, wpmm, strands=3)
    G = load_genome(g, cfg.frag_len, -1)
    got = map_reads_pssm(G, reads, lens, d_pssm, strands=3, variant=variant)
    _cmp(got, want, f"pssm variant {variant}")


@pytest.mark.parametrize("strands", [1, 2, 3])
@pytest.mark.parametrize("F,V", [(1000, 0), (1000, 17), (4096, -1), (300, -1), (50_000, -1), (100, -1)])
def test_pssm_geometries(oracle_mod, tiny, F, V, strands):
    from gpu_util import load_genome, map_reads_pssm, pssm_tables
    cfg, g, reads, lens, quals = tiny
    d_pssm, pm, pmm = pssm_tables(quals[:40], lens[:40])
    wpm, wpmm = oracle_mod.pssm_from_phred(quals[:40], 5, -4, 16)            # the oracle's own table feeds the oracle
    assert (pm == wpm).all() and (pmm == wpmm).all()
    want = oracle_mod.map_reads_pssm_parallel(g, F, V, reads[:40], lens[:40], wpm, wpmm, strands=strands)
    G = load_genome(g, F, V)
    got = map_reads_pssm(G, reads[:40], lens[:40], d_pssm, strands=strands)
    _cmp(got, want, f"pssm F={F} V={V} strands={strands}")


def test_pssm_ragged_lengths_and_long_reads(oracle_mod, tiny):
    from gpu_util import load_genome, map_reads_pssm, pssm_tables
    cfg, g, _, _, _ = tiny
    rng = np.random.default_rng(4343)
    n, M = 40, 250
    lens = rng.integers(1, M + 1, size=n).astype(np.int32)
    lens[:3] = [1, 2, M]
    reads = np.full((n, M), gen.N, dtype=np.uint8)
    for i in range(n):
        p = int(rng.integers(0, g.size - M))
        rd = g[p:p + lens[i]].copy()
        flip = rng.random(lens[i]) < 0.15
        rd[flip] = rng.integers(0, 5, size=int(flip.sum()))
        reads[i, :lens[i]] = gen.revcomp(rd) if i % 2 else rd
    quals = gen.make_quals(n, M, 77)
    d_pssm, pm, pmm = pssm_tables(quals, lens, scale=8)
    wpm, wpmm = oracle_mod.pssm_from_phred(quals, 5, -4, 8)
    valid = np.arange(M)[None, :] < lens[:, None]
    assert (pm[valid] == wpm[valid]).all() and (pmm[valid] == wpmm[valid]).all() and (pm[~valid] == 0).all()
    want = oracle_mod.map_reads_pssm_parallel(g, 2048, -1, reads, lens, wpm, wpmm, strands=3)
    G = load_genome(g, 2048, -1)
    _cmp(map_reads_pssm(G, reads, lens, d_pssm, strands=3, scale=8), want, "pssm ragged")


def test_pssm_uniform_table_equals_plain_scan(tiny):
    """GPU-only consistency: a table with the same pair everywhere must reproduce mss_map_reads bit for bit."""
    import torch
    from gpu_util import load_genome, map_reads, map_reads_pssm, to_dev
    cfg, g, reads, lens, _ = tiny
    w = np.uint32((5 & 0xFFFF) | ((-4 & 0xFFFF) << 16))
    d_pssm = to_dev(np.full(reads.shape, w, dtype=np.uint32))
    G = load_genome(g, cfg.frag_len, -1)
    a = map_reads(G, reads, lens, strands=3)
    import paper_1403_2136_b200 as mss
    b = map_reads_pssm(G, reads, lens, d_pssm, strands=3, bound=mss.Scoring(5, -4, -26))     # a hand-made table states its own range
    torch.cuda.synchronize()
    _cmp(b, a, "uniform table")


def test_nw_pssm_parity(oracle_mod, tiny):
    from gpu_util import load_genome, map_reads_pssm, nw_align_pssm, pssm_tables
    cfg, g, reads, lens, quals = tiny
    d_pssm, _, _ = pssm_tables(quals, lens)
    pm, pmm = oracle_mod.pssm_from_phred(quals, 5, -4, 16)                    # oracle inputs come from the oracle only
    G = load_genome(g, cfg.frag_len, -1)
    top2 = oracle_mod.map_reads_pssm_parallel(g, cfg.frag_len, -1, reads, lens, pm, pmm, strands=3)
    assert (map_reads_pssm(G, reads, lens, d_pssm, strands=3) == top2).all()
    want = oracle_mod.nw_align_pssm(g, cfg.frag_len, -1, reads, lens, top2, pm, pmm, 16 * -26)
    got = nw_align_pssm(G, reads, lens, top2, d_pssm)
    assert (got[0] == want[0]).all(), "score"
    assert (got[1] == want[1]).all(), "ref_pos"
    assert (got[3] == want[3]).all(), "n_cigar"
    for r in range(reads.shape[0]):
        assert (got[2][r, :got[3][r]] == want[2][r, :want[3][r]]).all(), f"cigar of read {r}"
    # cheap gaps (many I/D in optimal paths) and a longer read band
    want = oracle_mod.nw_align_pssm(g, cfg.frag_len, -1, reads[:60], lens[:60], top2[:60], pm[:60], pmm[:60], -40)
    import paper_1403_2136_b200 as mss
    import torch
    from gpu_util import to_dev
    rp, rn = gen.pack_reads(reads[:60], lens[:60])
    sc, pos, cig, nc = mss.mss_nw_align_pssm(G, to_dev(rp), to_dev(rn), to_dev(lens[:60]), int(reads.shape[1]),
                                             to_dev(np.ascontiguousarray(top2[:60])), d_pssm[:60].contiguous(),
                                             mss.Scoring(80, -64, -40), 30, None)
    torch.cuda.synchronize()
    sc, pos, cig, nc = sc.cpu().numpy(), pos.cpu().numpy(), cig.cpu().numpy().view(np.uint32), nc.cpu().numpy()
    assert (sc == want[0]).all() and (pos == want[1]).all() and (nc == want[3]).all()
    for r in range(60):
        assert (cig[r, :nc[r]] == want[2][r, :want[3][r]]).all(), f"cheap-gap cigar of read {r}"


def test_next_row_argument_errors(tiny):
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, to_dev
    cfg, g, reads, lens, quals = tiny
    G = load_genome(g, cfg.frag_len, -1)
    rp, rn = gen.pack_reads(reads[:4], lens[:4])
    d_q = to_dev(quals[:4])
    with pytest.raises(mss.MssError) as e:
        mss.mss_pssm_build(d_q, to_dev(lens[:4]), mss.Scoring(5, -4, -26), 10_000)         # 5*10000 > 32767
    assert e.value.status == -2
    d_p = mss.mss_pssm_build(d_q, to_dev(lens[:4]), mss.Scoring(5, -4, -26), 16)
    with pytest.raises(mss.MssError) as e:                                                   # 100 * 400 > 32767
        mss.mss_map_reads_pssm(G, to_dev(rp), to_dev(rn), to_dev(lens[:4]), 100, d_p, mss.Scoring(400, -320, -1000), 3)
    assert e.value.status == -2
    with pytest.raises(mss.MssError) as e:                                                   # table rows shorter than max_len
        mss.mss_map_reads_pssm(G, to_dev(rp), to_dev(rn), to_dev(lens[:4]), 100, d_p[:, :50].contiguous(),
                               mss.pssm_bound(mss.Scoring(), 16), 3)
    assert e.value.status == -1


def _pssm_fragment_scores(oracle_mod, g, F, V, q, m, pm, pmm):
    """Exact per-fragment PSSM scores of one strand-oriented query (q, pm, pmm already oriented): the pinned PSSM oracle on
    a genome cut to each fragment's readable window (one fragment, forward strand)."""
    nfrag = -(-g.size // F)
    out = np.zeros(nfrag, dtype=np.int64)
    veff = m - 1 if (V < 0 or V > m - 1) else V
    for f in range(nfrag):
        sub = g[f * F: min(g.size, f * F + F + veff)]
        padn = np.full(F + veff, gen.N, dtype=np.uint8); padn[:sub.size] = sub
        r = oracle_mod.map_reads_pssm(padn, F, veff, q[None, :m], [m], pm[None, :m], pmm[None, :m], strands=1)
        out[f] = r[0, 0, 2] if r[0, 0, 0] == 0 else (r[0, 1, 2] if r[0, 1, 0] == 0 else 0)
    return out


@pytest.mark.parametrize("F,V,m,scale", [(1000, -1, 100, 16), (1000, 0, 75, 16), (700, 30, 51, 8), (2048, -1, 150, 16)])
def test_pssm_pass1_bounds_hold(oracle_mod, F, V, m, scale):
    """Pass 1 under base-quality scoring (scan_filter_lq_kernel, PSSM form): u <= exact <= u + delta for every read, strand
    and fragment against the oracle's PSSM scores, reads with N, ragged lengths and Q2 tails included."""
    import torch
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, pssm_tables, to_dev
    g = gen.make_genome(24_000, 41)[0]
    g[3000:3200] = gen.N
    r = gen.make_reads(g, 20, m, 4100 + m, sub_rate=0.15)
    reads, lens = r["reads"].copy(), r["lens"].copy()
    lens[4] = m - 9; reads[4, lens[4]:] = gen.N
    lens[6] = 1; reads[6, 1:] = gen.N
    reads[2, m // 3] = gen.N
    reads[11, m // 2: m // 2 + 3] = gen.N
    quals = gen.make_quals(20, m, 4200 + m)
    d_pssm, _, _ = pssm_tables(quals, lens, scale=scale)
    pm, pmm = oracle_mod.pssm_from_phred(quals, 5, -4, scale)            # the oracle's own table feeds the oracle
    G = load_genome(g, F, V)
    rp, rn = gen.pack_reads(reads, lens)
    bound = mss.pssm_bound(mss.Scoring(), scale)
    u, delta = mss.mss_map_reads_bounds_pssm(G, to_dev(rp), to_dev(rn), to_dev(lens), m, d_pssm, bound, 3)
    torch.cuda.synchronize()
    u = u.cpu().numpy().view(np.uint16).astype(np.int64)
    assert delta == min(bound.match, -bound.mismatch) - bound.mismatch
    assert pm.max() <= bound.match and pmm.min() >= bound.mismatch       # the stated range holds for the oracle's table
    for i in range(reads.shape[0]):
        mi = int(lens[i])
        for s in (0, 1):
            q = gen.revcomp(reads[i, :mi]) if s else reads[i, :mi]
            a, b = (pm[i, :mi][::-1], pmm[i, :mi][::-1]) if s else (pm[i, :mi], pmm[i, :mi])
            ex = _pssm_fragment_scores(oracle_mod, g, F, V, q, mi, np.ascontiguousarray(a), np.ascontiguousarray(b))
            assert (u[i, s] != 0xFFFF).all()
            assert (u[i, s] <= ex).all() and (ex <= u[i, s] + delta).all(), (i, s, int(np.argmax(np.abs(ex - u[i, s]))))


def test_pssm_takes_the_two_pass_scan(oracle_mod, tiny):
    """The automatic PSSM scan is the two-pass scan (pass 1 in its PSSM form), with records identical to the oracle's; a
    read with an N and the tile kernel request (variant 13: no PSSM pass 1 there) fall back without changing the records."""
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, map_reads_pssm, pssm_tables
    cfg, g, reads, lens, quals = tiny
    reads = reads.copy()
    reads[3, 50] = gen.N
    d_pssm, _, _ = pssm_tables(quals, lens)
    wpm, wpmm = oracle_mod.pssm_from_phred(quals, 5, -4, 16)
    want = oracle_mod.map_reads_pssm_parallel(g, cfg.frag_len, -1, reads, lens, wpm, wpmm, strands=3)
    G = load_genome(g, cfg.frag_len, -1)
    got = map_reads_pssm(G, reads, lens, d_pssm, strands=3)
    info = mss.mss_get_last_launch()
    assert info["variant"] == 7 and info["pass1_kernel"] == 5
    _cmp(got, want, "pssm two-pass")
    _cmp(map_reads_pssm(G, reads, lens, d_pssm, strands=3, variant=13), want, "pssm, tile kernel requested")
    assert mss.mss_get_last_launch()["pass1_kernel"] == 0


def test_pssm_two_pass_chunk_loop(oracle_mod, tiny):
    """The two-pass scan works through the reads in chunks; every chunk must see ITS rows of the base-quality table (a chunk
    that read the first rows again would still produce plausible records).  1, 7 and 100 reads per chunk."""
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, map_reads_pssm, pssm_tables
    cfg, g, reads, lens, quals = tiny
    d_pssm, _, _ = pssm_tables(quals, lens)
    wpm, wpmm = oracle_mod.pssm_from_phred(quals, 5, -4, 16)
    want = oracle_mod.map_reads_pssm_parallel(g, cfg.frag_len, -1, reads, lens, wpm, wpmm, strands=3)
    G = load_genome(g, cfg.frag_len, -1)
    try:
        for nbytes in (20_000, 1400, 200):                # 50 fragments x 2 strands x 2 B = 200 B of bounds per read
            mss.mss_set_two_pass_chunk_bytes(nbytes)
            got = map_reads_pssm(G, reads, lens, d_pssm, strands=3)
            info = mss.mss_get_last_launch()
            assert info["variant"] == 7 and info["launches"] >= 2 * (reads.shape[0] * 200 // nbytes)
            _cmp(got, want, f"pssm chunk bytes {nbytes}")
    finally:
        mss.mss_set_two_pass_chunk_bytes(0)
