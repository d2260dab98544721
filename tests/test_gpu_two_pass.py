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


# pass-1 kernels and arithmetic: (scan variant, arithmetic of the lane-per-query kernel)
#   (7, -1) automatic = lane-per-query kernel, e5m2 operand bytes where the scoring allows; (7, 0) packed int16 DPX;
#   (7, 1) fp16 pairs; (7, 2) e5m2 bytes (lowered where the scoring is not exact in e5m2); (13, -1) the tile kernel
#   (7, 8) / (7, 10) int16 / e5m2 arithmetic with the plane offsets read from the shared-memory table instead of registers
PASS1 = [(7, -1), (7, 0), (7, 1), (7, 2), (7, 8), (7, 10), (13, -1)]


class pass1_setup:
    """Select the pass-1 kernel for the calls inside the with-block (thread-local switches of the library)."""

    def __init__(self, variant=7, arithmetic=-1, query_sets=0, tile=0):
        self.args = (variant, arithmetic, query_sets, tile)

    def __enter__(self):
        import paper_1403_2136_b200 as mss
        v, a, q, t = self.args
        mss.mss_set_pass1_geometry(q, t, a)
        mss.mss_set_scan_variant(v)
        return self

    def __exit__(self, *exc):
        import paper_1403_2136_b200 as mss
        mss.mss_set_pass1_geometry(0, 0, -1)
        mss.mss_set_scan_variant(0)


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
    """Every pass-1 kernel and arithmetic: u <= exact <= u + delta against the oracle's per-fragment scores; the
    bounds of the different kernels are the same integers (they compute the same recurrence).  Reads holding an N are
    bounded too by the lane-per-query kernel (N planes); the tile kernel leaves them at 0xFFFF."""
    from gpu_util import load_genome
    g = gen.make_genome(40_000, 31)[0]
    g[5000:5300] = gen.N
    r = gen.make_reads(g, 24, m, 3100 + m, sub_rate=0.15)
    reads, lens = r["reads"], r["lens"].copy()
    lens[5] = max(1, m - 7); reads[5, lens[5]:] = gen.N
    lens[9] = 1; reads[9, 1:] = gen.N
    with_n = [2, 13, 17]
    reads[2, m // 3] = gen.N                               # one N
    reads[13, 0] = gen.N; reads[13, m - 1] = gen.N         # first and last position
    reads[17, m // 2: m // 2 + 3] = gen.N                  # a run: (c, N), (N, N), (N, c) double steps whatever the parity
    G = load_genome(g, F, V)
    exact = {(i, s): _exact_fragment_scores(oracle_mod, g, F, V, reads[i], int(lens[i]), s, match, mismatch, fast)
             for i in range(reads.shape[0]) for s in (0, 1)}
    first = None
    for variant, arith in PASS1:
        with pass1_setup(variant, arith):
            u, delta = _bounds(G, reads, lens, 3, match, mismatch, fast)
        assert delta == min(match, -mismatch) - mismatch
        for (i, s), ex in exact.items():
            ui = u[i, s]
            if variant == 13 and i in with_n and (ui == 0xFFFF).all():
                continue                                    # the tile kernel does not scan reads with an N on a scored position
            assert (ui != 0xFFFF).all(), (variant, arith, i, s)
            assert (ui <= ex).all() and (ex <= ui + delta).all(), (variant, arith, i, s, int(np.argmax(np.abs(ex - ui))))
        if first is None:
            first = u
        same = (u != 0xFFFF) & (first != 0xFFFF)
        assert (u[same] == first[same]).all(), (variant, arith)


def test_pass1_reads_with_n(oracle_mod):
    """A read with an N: the lane-per-query kernel switches the block to the tile with the N planes and bounds it like any
    other read; the tile kernel marks it unbounded (0xFFFF = every fragment is a candidate).  Either way the other reads of
    the block are unaffected, and a block without N reads keeps the large tile."""
    from gpu_util import load_genome
    g = gen.make_genome(20_000, 32)[0]
    r = gen.make_reads(g, 40, 60, 3200, sub_rate=0.1)
    reads, lens = r["reads"].copy(), r["lens"]
    clean, _ = None, None
    G = load_genome(g, 1000, -1)
    with pass1_setup(7, -1):
        clean, _ = _bounds(G, reads, lens, 3)
    reads[2, 17] = gen.N
    with pass1_setup(7, -1):
        u, delta = _bounds(G, reads, lens, 3)
    assert (u != 0xFFFF).all()
    keep = np.arange(40) != 2
    assert (u[keep] == clean[keep]).all()                   # same bounds through the other tile geometry
    for s in (0, 1):
        ex = oracle_mod.fragment_scores(g, 1000, -1, reads[2], strand=s, opt="O3")[0]
        assert (u[2, s] <= ex).all() and (ex <= u[2, s] + delta).all()
    with pass1_setup(13, -1):
        ut, _ = _bounds(G, reads, lens, 3)
    assert (ut[2] == 0xFFFF).all() and (ut[keep] == clean[keep]).all()


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
    want_fast = oracle_mod.map_reads_parallel(g, F, V, reads, lens, strands=strands, fast=True)
    for variant, arith in PASS1:
        with pass1_setup(variant, arith):
            _cmp(map_reads(G, reads, lens, strands=strands, variant=variant), want, f"two-pass {variant}/{arith} F={F} V={V} strands={strands}")
        with pass1_setup(variant, arith):
            _cmp(map_reads_fast(G, reads, lens, strands=strands, variant=variant), want_fast,
                 f"two-pass fast {variant}/{arith} F={F} V={V} strands={strands}")


@pytest.mark.parametrize("m", [1, 2, 3, 35, 36, 37, 52, 53, 60, 64, 65, 76, 77, 100, 101, 127, 128, 129, 152, 153, 159, 160, 161, 255, 256, 257,
                               300, 409, 600])
def test_two_pass_read_lengths_across_the_register_table_limits(oracle_mod, m):
    """The lane-per-query pass 1 keeps a query's plane offsets in registers: 32, 64 or 80 double steps directly, up to 128
    as 16-bit pairs; longer reads read them from the shared-memory table (and the longest take the tile kernel).  Lengths on
    both sides of every limit, mixed with shorter reads in the same block (padding steps on the all-zero plane), all three
    arithmetics, offsets in registers and from the table, 8 and 16 chains per thread (the 16-chain instances serve 1-52 and
    65-76 scored positions: lengths on both sides of those limits too)."""
    from gpu_util import load_genome, map_reads
    g = gen.make_genome(30_000, 36)[0]
    r = gen.make_reads(g, 40, m, 3600 + m, sub_rate=0.12, indel_prob=0.0 if m < 8 else 0.5)
    reads, lens = r["reads"].copy(), r["lens"].copy()
    for k, short in ((3, m // 2), (8, m - 1), (20, 1), (21, 2)):
        if 1 <= short < m:
            lens[k] = short; reads[k, short:] = gen.N
    G = load_genome(g, 1536, -1)
    want = oracle_mod.map_reads_parallel(g, 1536, -1, reads, lens, strands=3)
    for arith in (-1, 0, 1, 2, 8, 9, 10, 34):
        with pass1_setup(7, arith):
            _cmp(map_reads(G, reads, lens, strands=3, variant=7), want, f"m={m} arithmetic {arith}")


@pytest.mark.parametrize("query_sets,tile", [(1, 0), (2, 0), (4, 0), (1, 512), (2, 1024), (4, 768), (1, 2048)])
def test_pass1_reads_per_block_and_tile_do_not_change_results(oracle_mod, query_sets, tile):
    """BASELINE.json config 5's "reads-per-block swept": 16, 32 or 64 reads (x 2 strands) per block, and forced tiles
    including ragged ones (F = 1000 is not a multiple of any tile), partial last groups (75 reads)."""
    from gpu_util import load_genome, map_reads
    import paper_1403_2136_b200 as mss
    cfg = gen.config(1)
    g, _ = cfg.genome()
    r = cfg.reads(g)
    reads, lens = r["reads"][:75].copy(), r["lens"][:75].copy()
    reads[1::2] = np.stack([gen.revcomp(x) for x in reads[1::2]])
    for F in (1000, 4096):
        G = load_genome(g, F, -1)
        want = oracle_mod.map_reads_parallel(g, F, -1, reads, lens, strands=3)
        for strands in (1, 3):
            w = want if strands == 3 else oracle_mod.map_reads_parallel(g, F, -1, reads, lens, strands=1)
            with pass1_setup(7, -1, query_sets, tile):
                got = map_reads(G, reads, lens, strands=strands, variant=7)
                info = mss.mss_get_last_launch()
            _cmp(got, w, f"query_sets={query_sets} tile={tile} F={F} strands={strands}")
            assert info["variant"] == 7 and info["reads_per_block"] == 32 * query_sets // (2 if strands == 3 else 1)
            assert info["pass1_kernel"] == 4                             # lane-per-query kernel, e5m2 operands (5/-4 scoring)
            if tile:
                assert info["tile_diagonals"] == tile


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
        for variant, arith in PASS1:
            with pass1_setup(variant, arith):
                _cmp(map_reads(G, reads, lens, strands=3, variant=variant), want, f"ties {variant}/{arith}")
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
        for variant, arith in PASS1:
            with pass1_setup(variant, arith):
                _cmp(map_reads(G, r["reads"], r["lens"], match=match, mismatch=mismatch, variant=variant), want,
                     f"scoring {match}/{mismatch} pass 1 {variant}/{arith}")
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
