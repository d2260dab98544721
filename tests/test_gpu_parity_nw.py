"""-m gpu: the CUDA Needleman-Wunsch stage against the oracle: score, position, CIGAR -- bit-exact."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


def _check(oracle_mod, g, F, V, reads, lens, strands=3, pad=30, gap=-26, match=5, mismatch=-4, cigar_stride=None):
    from gpu_util import load_genome, nw_align
    top2 = oracle_mod.map_reads_parallel(g, F, V, reads, lens, match=match, mismatch=mismatch, strands=strands)
    want = oracle_mod.nw_align(g, F, V, reads, lens, top2, match=match, mismatch=mismatch, gap=gap, pad=pad,
                               cigar_stride=cigar_stride)
    G = load_genome(g, F, V)
    got = nw_align(G, reads, lens, top2, match=match, mismatch=mismatch, gap=gap, pad=pad, cigar_stride=cigar_stride)
    assert (got[0] == want[0]).all(), np.where(got[0] != want[0])[0][:5]
    assert (got[1] == want[1]).all(), np.where(got[1] != want[1])[0][:5]
    assert (got[3] == want[3]).all(), np.where(got[3] != want[3])[0][:5]
    stride = got[2].shape[1]
    for k in range(len(lens)):
        n = min(int(want[3][k]), stride)
        assert (got[2][k, :n] == want[2][k, :n]).all(), (k, got[2][k, :n], want[2][k, :n])


def test_tiny_config(oracle_mod):
    cfg = gen.config(1)
    g, _ = cfg.genome()
    r = cfg.reads(g)
    _check(oracle_mod, g, cfg.frag_len, cfg.overlap, r["reads"], r["lens"], strands=3)


@pytest.mark.parametrize("m", [1, 5, 31, 32, 33, 36, 51, 64, 100, 150, 250, 257, 300, 700])
def test_read_lengths_and_bands(oracle_mod, m):
    g = gen.make_genome(30_000, 31)[0]
    r = gen.make_reads(g, 24, m, 1000 + m, sub_rate=(0.05, 0.3))
    _check(oracle_mod, g, 2048, -1, r["reads"], r["lens"])


def test_mixed_lengths_cheap_gaps_and_n(oracle_mod):
    g = gen.make_genome(20_000, 32)[0].copy()
    g[5000:5100] = gen.N
    rs = [gen.make_reads(g, 12, m, 2000 + m, sub_rate=0.15) for m in (40, 90, 130)]
    ml = 130
    reads = np.full((36, ml), gen.N, dtype=np.uint8)
    lens = np.zeros(36, dtype=np.int32)
    for k, r in enumerate(rs):
        mm = r["reads"].shape[1]
        reads[12 * k:12 * k + 12, :mm] = r["reads"]
        lens[12 * k:12 * k + 12] = mm
    reads[3, 7] = gen.N
    for gap in (-26, -6, -1):
        _check(oracle_mod, g, 1000, 20, reads, lens, gap=gap, pad=10)
    _check(oracle_mod, g, 1000, -1, reads, lens, gap=-3, pad=0, cigar_stride=3)


def test_tiny_windows_and_genome_edges(oracle_mod):
    g = gen.make_genome(300, 33)[0]
    reads = np.stack([g[0:40], g[260:300], gen.revcomp(g[100:140]), g[10:50]])
    lens = np.full(4, 40, dtype=np.int32)
    _check(oracle_mod, g, 64, -1, reads, lens)
    _check(oracle_mod, g, 16, 0, reads, lens, pad=0)       # window shorter than the read: forced insertions
    _check(oracle_mod, g, 300, -1, reads, lens)
