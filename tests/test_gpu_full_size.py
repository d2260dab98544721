"""-m gpu: BASELINE.json's configs at their full geometry, in the launch configuration bench.py times.  The oracle cannot
finish 1e13+ cells in seconds, so it checks a seeded sample of reads one by one (all fragments, both strands, top-2 and NW),
plus properties that hold at any size for every read."""
import os

import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


def _device_inputs(genome, reads, lens):
    from gpu_util import to_dev
    rp, rn = gen.pack_reads(reads, lens)
    return to_dev(rp), to_dev(rn), to_dev(lens)


def _properties(top2, lens, n_frag, F, match=5):
    best, second = top2[:, 0], top2[:, 1]
    assert (best[:, 0] >= 0).all() and (best[:, 0] < n_frag).all()
    assert ((second[:, 0] >= 0) & (second[:, 0] < n_frag) & (second[:, 0] != best[:, 0])).all()
    assert (best[:, 1] >= 0).all() and (best[:, 1] < F).all() and (second[:, 1] >= 0).all() and (second[:, 1] < F).all()
    assert (best[:, 2] >= second[:, 2]).all() and (second[:, 2] >= 0).all() and (best[:, 2] <= match * lens).all()
    tie = best[:, 2] == second[:, 2]
    assert (best[tie, 0] < second[tie, 0]).all()                       # ties keep the lowest fragment first
    assert set(np.unique(top2[:, :, 3])) <= {0, 1}


def _sample_check(oracle_mod, genome, cfg, reads, lens, top2, nw, idx):
    want = oracle_mod.map_reads_parallel(genome, cfg.frag_len, cfg.overlap, reads[idx], lens[idx], strands=cfg.strands)
    bad = np.where((top2[idx] != want).any(axis=(1, 2)))[0]
    assert bad.size == 0, (idx[bad[0]], top2[idx][bad[0]].tolist(), want[bad[0]].tolist())
    ws, wp, wc, wn = oracle_mod.nw_align(genome, cfg.frag_len, cfg.overlap, reads[idx], lens[idx], want, cigar_stride=64)
    score, pos, cigar, ncig = nw
    assert (score[idx] == ws).all() and (pos[idx] == wp).all() and (ncig[idx] == wn).all()
    for k, i in enumerate(idx):
        n = min(int(wn[k]), cigar.shape[1], 64)
        assert (cigar[i, :n] == wc[k, :n]).all(), (i, cigar[i, :n], wc[k, :n])


def _run(cfg, genome, reads, lens, cigar_stride=32):
    import torch
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome
    G = load_genome(genome, cfg.frag_len, cfg.overlap)
    d_reads, d_mask, d_lens = _device_inputs(genome, reads, lens)
    m = int(reads.shape[1])
    top2 = mss.mss_map_reads(G, d_reads, d_mask, d_lens, m, mss.Scoring(), cfg.strands)
    sc, pos, cig, nc = mss.mss_nw_align(G, d_reads, d_mask, d_lens, m, top2, mss.Scoring(), 30, cigar_stride)
    torch.cuda.synchronize()
    info = mss.mss_get_last_launch()
    return G, top2.cpu().numpy(), (sc.cpu().numpy(), pos.cpu().numpy(), cig.cpu().numpy().view(np.uint32), nc.cpu().numpy()), info


def _truth_rate(cfg, r, top2):
    """Reported, not asserted bit-for-bit: top-1 fragment within +-1 of the true fragment."""
    true_frag = r["start"] // cfg.frag_len
    return float(np.mean(np.abs(top2[:, 0, 0] - true_frag) <= 1))


def test_config2_full_100k_reads(oracle_mod):
    cfg = gen.config(2)
    genome, _ = cfg.genome()
    r = cfg.reads(genome)
    G, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"])
    assert top2.shape == (100_000, 2, 4) and G.n_frag == 1124
    _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 22))
    idx = np.sort(rng.choice(100_000, size=4 * (os.cpu_count() or 8), replace=False))
    _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], top2, nw, idx)
    assert _truth_rate(cfg, r, top2) > 0.9                              # sanity of the workload, not parity


def test_config3_length_sweep_geometry(oracle_mod):
    cfg = gen.config(3)
    genome, _ = cfg.genome()
    r = cfg.reads(genome, limit=256)                                    # 15 groups x 256 reads, lengths 36..250 in one call
    G, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"], cigar_stride=64)
    _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 32))
    idx = np.sort(np.concatenate([g * 256 + rng.choice(256, size=3, replace=False) for g in range(15)]))
    _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], top2, nw, idx)


def test_config5_throughput_geometry(oracle_mod):
    cfg = gen.config(5)
    genome, _ = cfg.genome()
    r = cfg.reads(genome, limit=20_000)
    G, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"])
    _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 52))
    idx = np.sort(rng.choice(20_000, size=2 * (os.cpu_count() or 8), replace=False))
    _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], top2, nw, idx)


@pytest.mark.skipif(os.environ.get("MSS_SKIP_CHR1") == "1", reason="MSS_SKIP_CHR1=1")
def test_config4_chr1_sized_genome(oracle_mod):
    """249 Mbp with N runs and planted duplicates, F = 16384: the genome no longer fits L2 tiles of one block range."""
    cfg = gen.config(4)
    genome, info_g = cfg.genome()
    r = cfg.reads(genome, limit=384)
    G, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"], cigar_stride=64)
    assert G.n_frag == 15_198
    _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
    # reads drawn inside a planted duplicate must see the other copy as a strong second place
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 42))
    idx = np.sort(rng.choice(384, size=max(4, (os.cpu_count() or 8) // 2), replace=False))
    _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], top2, nw, idx)
