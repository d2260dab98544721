"""T1: the seeded generators and the wire format (gen/) -- determinism, round trips, recipe shapes."""
import numpy as np

import gen


def test_pack_roundtrip_and_bit_layout():
    codes = gen.encode("ACGTNACGTTTGACNNA")
    packed, nmask = gen.pack_2bit(codes)
    assert packed.dtype == np.uint32 and packed.size == 2 and nmask.size == 1
    # base i in bits [2*(i%16), +2) of word i//16, A=0 C=1 G=2 T=3; N -> code 0 + mask bit
    assert packed[0] & 0xFF == (0 | 1 << 2 | 2 << 4 | 3 << 6)
    assert (nmask[0] >> 4) & 1 == 1 and (nmask[0] >> 14) & 3 == 3 and nmask[0] & 0xF == 0
    assert (gen.unpack_2bit(packed, nmask, codes.size) == codes).all()
    rng = np.random.default_rng(0)
    big = rng.integers(0, 5, size=100_003).astype(np.uint8)
    p, n = gen.pack_2bit(big)
    assert (gen.unpack_2bit(p, n, big.size) == big).all()


def test_pack_reads_layout():
    rng = np.random.default_rng(1)
    reads = rng.integers(0, 5, size=(9, 53)).astype(np.uint8)
    lens = rng.integers(1, 54, size=9).astype(np.int32)
    p, n = gen.pack_reads(reads, lens)
    assert p.shape == (9, 4) and n.shape == (9, 2)
    for r in range(9):
        got = gen.unpack_2bit(p[r], n[r], int(lens[r]))
        assert (got == reads[r, :lens[r]]).all()
        # bits beyond the length are zero
        full = gen.unpack_2bit(p[r], n[r], 64)
        assert (full[lens[r]:] == 0).all()
    p8, n8 = gen.pack_reads(reads, lens, stride_words=8)
    assert p8.shape == (9, 8) and (p8[:, :4] == p).all() and (p8[:, 4:] == 0).all()


def test_revcomp():
    assert gen.decode(gen.revcomp(gen.encode("AACGTN"))) == "NACGTT"


def test_determinism_and_hashes():
    cfg = gen.config(1)
    g1, _ = cfg.genome()
    g2, _ = cfg.genome()
    r1, r2 = cfg.reads(g1), cfg.reads(g2)
    assert gen.sha256_of(g1) == gen.sha256_of(g2)
    assert gen.sha256_of(r1["reads"], r1["lens"]) == gen.sha256_of(r2["reads"], r2["lens"])
    assert g1.size == 50_000 and r1["reads"].shape == (200, 100) and (r1["strand"] == 0).all()
    assert set(np.unique(g1)) == {0, 1, 2, 3}
    # about half of the Tiny reads carry one indel (recipe: p = 0.5)
    assert 60 <= int(r1["n_indel"].sum()) <= 140


def test_read_recipe_statistics():
    g, _ = gen.make_genome(200_000, 5)
    r = gen.make_reads(g, 4000, 100, 6, sub_rate=(0.10, 0.30), both_strands=True)
    assert abs(r["strand"].mean() - 0.5) < 0.05
    assert 0.10 <= r["p"].min() and r["p"].max() <= 0.30
    plain = (r["n_indel"] == 0)
    fwd = plain & (r["strand"] == 0)
    idx = np.where(fwd)[0][:300]
    ident = np.array([(r["reads"][i] == g[r["start"][i]:r["start"][i] + 100]).mean() for i in idx])
    assert abs((1 - ident).mean() - 0.20) < 0.02          # mean substitution rate of U[0.1, 0.3]
    rev = np.where(plain & (r["strand"] == 1))[0][:300]
    ident = np.array([(gen.revcomp(r["reads"][i]) == g[r["start"][i]:r["start"][i] + 100]).mean() for i in rev])
    assert abs((1 - ident).mean() - 0.20) < 0.02
    assert (r["span"][plain] == 100).all()
    assert (np.abs(r["span"] - 100) <= 60).all() and (r["start"] + r["span"] <= g.size).all()


def test_config4_recipe_small():
    g, info = gen.make_genome(3_000_000, 9, gc=0.41, dup_frac=0.02, n_frac=0.10)
    assert abs((g == gen.N).mean() - 0.10) < 0.005
    acgt = g[g < 4]
    assert abs(((acgt == gen.C) | (acgt == gen.G)).mean() - 0.41) < 0.01
    assert sum(d[2] for d in info["dups"]) >= 0.02 * g.size * 0.99
    r = gen.make_reads(g, 500, 150, 10, sub_rate=0.20, avoid_n=True)
    for i in range(500):
        assert (g[r["start"][i]:r["start"][i] + r["span"][i]] < 4).all()


def test_cells_formula():
    cfg = gen.config(2)
    assert cfg.cells() == 100_000 * 100 * 1124 * 4096 * 2
    assert gen.config(1).cells() == 200 * 100 * 50 * 1000


def test_quals_are_seeded_and_in_range():
    """gen.make_quals: same seed -> same bytes; phred values in [2, 41]; a share of reads carries a Q2 tail."""
    a = gen.make_quals(500, 100, 123)
    b = gen.make_quals(500, 100, 123)
    c = gen.make_quals(500, 100, 124)
    assert a.dtype == np.uint8 and a.shape == (500, 100)
    assert (a == b).all() and (a != c).any()
    assert a.min() >= 2 and a.max() <= 41
    tails = (a[:, -1] == 2).mean()
    assert 0.05 < tails < 0.3


def test_chunked_packing_equals_one_shot(monkeypatch):
    """pack_2bit works chunk by chunk for Gbp-sized genomes: any chunk size gives the same words."""
    from gen import synth
    rng = np.random.default_rng(9)
    codes = rng.integers(0, 5, size=200_003).astype(np.uint8)
    whole = gen.pack_2bit(codes)
    monkeypatch.setattr(synth, "_PACK_CHUNK", 4096)
    parts = gen.pack_2bit(codes)
    assert (whole[0] == parts[0]).all() and (whole[1] == parts[1]).all()
    assert (gen.unpack_2bit(parts[0], parts[1], codes.size) == codes).all()


def test_config6_is_the_table8_shape():
    """PAPER.md:182, Table 8: 76 bp reads against a 2.4 Gbp genome, fragment length 4800."""
    cfg = gen.config(6)
    assert (cfg.genome_len, cfg.frag_len, cfg.max_len, cfg.strands) == (2_400_000_000, 4800, 76, 3)
    assert -(-cfg.genome_len // cfg.frag_len) == 500_000
