"""-m gpu: edge and degenerate cases of the MaxSS scan against the oracle, bit-exact (tier T2)."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


def _cmp(got, want, ctx=""):
    bad = np.where((got != want).any(axis=(1, 2)))[0]
    assert bad.size == 0, f"{ctx}: {bad.size} reads differ, first {bad[0]}: got {got[bad[0]].tolist()} want {want[bad[0]].tolist()}"


def _both(oracle_mod, g, F, V, reads, lens, strands=3, variants=(0, 1), **kw):
    from gpu_util import load_genome, map_reads
    want = oracle_mod.map_reads_parallel(g, F, V, reads, lens, strands=strands,
                                         **{k: v for k, v in kw.items() if k in ("match", "mismatch")})
    G = load_genome(g, F, V)
    for v in variants:
        got = map_reads(G, reads, lens, strands=strands, variant=v, **kw)
        _cmp(got, want, f"F={F} V={V} strands={strands} variant={v}")
    return want


def test_empty_batch_and_bad_lengths(oracle_mod):
    import torch
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, to_dev
    g = gen.make_genome(5000, 5)[0]
    G = load_genome(g, 512, -1)
    out = mss.mss_map_reads(G, torch.zeros((0, 4), dtype=torch.int32, device="cuda"), None,
                            torch.zeros(0, dtype=torch.int32, device="cuda"), 50)
    assert out.shape == (0, 2, 4)
    # lengths outside [1, max_len] -> no fragment for that read; neighbours unaffected
    r = gen.make_reads(g, 6, 50, 6, sub_rate=0.1)
    lens = r["lens"].copy()
    lens[1] = 0
    lens[4] = 51
    rp, rn = gen.pack_reads(r["reads"], np.clip(lens, 0, 50))
    got = mss.mss_map_reads(G, to_dev(rp), to_dev(rn), to_dev(lens), 50).cpu().numpy()
    torch.cuda.synchronize()
    want = oracle_mod.map_reads(g, 512, -1, r["reads"], r["lens"], strands=3)
    for k in range(6):
        if k in (1, 4):
            assert got[k].tolist() == [[-1, 0, 0, 0], [-1, 0, 0, 0]]
        else:
            assert (got[k] == want[k]).all()


def test_all_n_read_all_n_genome_and_score_zero(oracle_mod):
    g = gen.make_genome(6000, 7)[0]
    reads = np.stack([np.full(64, gen.N, dtype=np.uint8),                       # all-N read: every fragment scores 0
                      g[100:164].copy()])
    lens = np.array([64, 64], dtype=np.int32)
    want = _both(oracle_mod, g, 700, -1, reads, lens)
    assert want[0].tolist() == [[0, 0, 0, 0], [1, 0, 0, 0]]                     # a fragment scoring 0 is still a fragment
    gn = np.full(3000, gen.N, dtype=np.uint8)                                   # all-N genome
    _both(oracle_mod, gn, 512, -1, reads, lens)
    # read over {A}, genome over {C,G,T}: nothing matches anywhere
    ga = (1 + gen.make_genome(4000, 8)[0] % 3).astype(np.uint8)
    _both(oracle_mod, ga, 1000, 0, np.zeros((1, 30), dtype=np.uint8), np.array([30], dtype=np.int32), strands=1)


@pytest.mark.parametrize("m", [1, 2, 3, 4, 5, 15, 16, 17, 33])
def test_very_short_reads(oracle_mod, m):
    g = gen.make_genome(9000, 9)[0]
    r = gen.make_reads(g, 10, m, 90 + m, sub_rate=0.0, indel_counts=(0,))
    _both(oracle_mod, g, 1024, -1, r["reads"], r["lens"])
    _both(oracle_mod, g, 300, 0, r["reads"], r["lens"], variants=(0,))


def test_one_and_two_fragments_and_ragged_last(oracle_mod):
    g = gen.make_genome(10_000, 10)[0]
    r = gen.make_reads(g, 12, 80, 11, sub_rate=0.15)
    for F in (10_000, 20_000, 5_000, 9_999, 5_001, 3_333, 257, 256, 255, 64, 7, 1):
        _both(oracle_mod, g, F, -1, r["reads"][:6] if F < 64 else r["reads"], r["lens"][:6] if F < 64 else r["lens"],
              variants=(0,))
    # every DPX tile size on a fragment length that is no multiple of anything
    for v in (2, 3, 4, 5, 6):
        _both(oracle_mod, g, 1777, 13, r["reads"], r["lens"], variants=(v,))


def test_ties_duplicates_palindromes_periodic(oracle_mod):
    rng = np.random.Generator(np.random.PCG64(12))
    g = gen.make_genome(12_000, 12)[0].copy()
    block = g[3 * 1000 + 100:3 * 1000 + 400].copy()
    g[7 * 1000 + 250:7 * 1000 + 550] = block                                    # identical copies in fragments 3 and 7
    read = block[50:150].copy()
    pal = np.concatenate([block[:30], gen.revcomp(block[:30])])                 # palindromic read: equals its own reverse complement
    reads = np.full((3, 100), gen.N, dtype=np.uint8)
    reads[0] = read
    reads[1, :60] = pal
    reads[2] = gen.revcomp(read)
    lens = np.array([100, 60, 100], dtype=np.int32)
    want = _both(oracle_mod, g, 1000, -1, reads, lens, variants=(0, 1, 3, 5))
    assert want[0, 0, 0] == 3 and want[0, 1, 0] == 7 and want[0, 0, 2] == want[0, 1, 2] == 500
    assert want[1, 0, 3] == 0 and want[2, 0, 3] == 1
    gp = np.tile(np.array([0, 1], dtype=np.uint8), 4000)                        # periodic genome ACAC...: lowest window start wins
    rp = np.tile(np.array([0, 1], dtype=np.uint8), 20)[None, :]
    wantp = _both(oracle_mod, gp, 1500, -1, rp, np.array([40], dtype=np.int32), variants=(0, 1, 2, 4))
    assert wantp[0, 0].tolist()[:3] == [0, 0, 200] and wantp[0, 1, 0] == 1
    del rng


def test_n_runs_in_genome_and_reads_mask_optional(oracle_mod):
    from gpu_util import load_genome, map_reads
    g = gen.make_genome(20_000, 13)[0].copy()
    g[4000:4700] = gen.N
    g[9990:10_010] = gen.N
    r = gen.make_reads(g, 24, 70, 14, sub_rate=0.1, avoid_n=True)        # N-free reads: the mask is optional for these
    assert (r["reads"] < 4).all()
    reads = r["reads"].copy()
    reads[3, 10:14] = gen.N
    reads[5, 0] = gen.N
    reads[6, 69] = gen.N
    _both(oracle_mod, g, 2048, -1, reads, r["lens"])
    # without an N mask the library must treat every read base as its 2-bit code
    want = oracle_mod.map_reads_parallel(g, 2048, -1, r["reads"], r["lens"], strands=3)
    G = load_genome(g, 2048, -1)
    got = map_reads(G, r["reads"], r["lens"], with_mask=False)
    _cmp(got, want, "no mask")
    got = map_reads(G, r["reads"], r["lens"], stride_words=9)                   # stride larger than needed
    _cmp(got, want, "stride 9")


def test_mixed_lengths_in_one_batch(oracle_mod):
    g = gen.make_genome(30_000, 15)[0]
    ms = (36, 51, 100, 150, 250)
    n = 8
    reads = np.full((n * len(ms), 250), gen.N, dtype=np.uint8)
    lens = np.zeros(n * len(ms), dtype=np.int32)
    for k, m in enumerate(ms):
        r = gen.make_reads(g, n, m, 150 + m, sub_rate=0.2)
        reads[k * n:(k + 1) * n, :m] = r["reads"]
        lens[k * n:(k + 1) * n] = m
    perm = np.random.Generator(np.random.PCG64(16)).permutation(lens.size)
    _both(oracle_mod, g, 4096, -1, reads[perm], lens[perm], variants=(0, 2, 3))
    _both(oracle_mod, g, 4096, 40, reads[perm], lens[perm], variants=(0,))       # explicit overlap shorter than most reads


@pytest.mark.parametrize("m", [700, 2432, 6553])
def test_long_reads_up_to_the_s16_limit(oracle_mod, m):
    """2432 = the paper's maximum read length; 6553 = floor(32767/5), this library's."""
    g = gen.make_genome(40_000, 17)[0]
    r = gen.make_reads(g, 3, m, 170 + m, sub_rate=0.05, indel_counts=(0, 1))
    reads = r["reads"].copy()
    reads[0] = g[1000:1000 + m]                                                 # exact read: score m*match, the s16 extreme
    want = _both(oracle_mod, g, 8192, -1, reads, r["lens"], variants=(0,))
    assert want[0, 0].tolist() == [0, 1000, 5 * m, 0]
    import paper_1403_2136_b200 as mss
    info = mss.mss_get_last_launch()
    assert info["variant"] != 1, info           # the tile kernel (fewer reads per block), not the generic fallback


def test_long_reads_several_groups_all_modes(oracle_mod):
    """m = 1500: 16 queries per block instead of 32, so 11 reads span two read groups; plain, fast and PSSM scans."""
    from gpu_util import load_genome, map_reads, map_reads_fast, map_reads_pssm, pssm_tables
    m, n = 1500, 11
    g = gen.make_genome(30_000, 21)[0]
    r = gen.make_reads(g, n, m, 2100, sub_rate=0.1, indel_counts=(0, 1, 2))
    reads, lens = r["reads"], r["lens"].copy()
    lens[3], lens[7] = 1499, 801
    reads[3, 1499:] = gen.N
    reads[7, 801:] = gen.N
    G = load_genome(g, 4096, -1)
    _cmp(map_reads(G, reads, lens), oracle_mod.map_reads_parallel(g, 4096, -1, reads, lens, strands=3), "plain m=1500")
    _cmp(map_reads_fast(G, reads, lens), oracle_mod.map_reads_parallel(g, 4096, -1, reads, lens, strands=3, fast=True), "fast m=1500")
    quals = gen.make_quals(n, m, 2101)
    d_pssm, _, _ = pssm_tables(quals, lens, scale=4)
    pm, pmm = oracle_mod.pssm_from_phred(quals, 5, -4, 4)                     # the oracle's own table
    _cmp(map_reads_pssm(G, reads, lens, d_pssm, scale=4),
         oracle_mod.map_reads_pssm_parallel(g, 4096, -1, reads, lens, pm, pmm, strands=3), "pssm m=1500")


def test_other_scorings_and_range_errors(oracle_mod):
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, map_reads
    g = gen.make_genome(15_000, 18)[0]
    r = gen.make_reads(g, 10, 90, 19, sub_rate=0.2)
    for match, mismatch in ((1, -1), (2, -3), (9, -7), (10, -40), (127, -128), (300, -1)):
        _both(oracle_mod, g, 1500, -1, r["reads"], r["lens"], match=match, mismatch=mismatch)
    G = load_genome(g, 1500, -1)
    for match, mismatch in ((0, -4), (5, 0), (5, 4), (400, -4)):               # 400*90 > 32767
        with pytest.raises(mss.MssError) as e:
            map_reads(G, r["reads"], r["lens"], match=match, mismatch=mismatch)
        assert e.value.status == -2
