"""-m gpu: BASELINE.json's configs at their full geometry, in the launch configuration bench.py times.  The oracle cannot
finish 1e13+ cells in seconds, so it checks a seeded sample of reads one by one (all fragments, both strands, top-2, NW and
the repeat filter) PLUS the reads where a pruning scan is most likely to go wrong -- those whose device record is a tie
(best = second) or a near-repeat (10*second >= 9*best) -- plus properties that hold at any size for every read.
Sample sizes scale with the host cores of the GPU box (SURVEY.md 8(d) "Oracle timing and coverage"); at 16 cores the
oracle work of this file is about 5 minutes."""
import os

import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu

CORES = os.cpu_count() or 8


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


def _repeat_like(top2, cap, seed):
    """Indices of reads whose device record is a tie or has second >= 0.9 * best (the repeat cases), at most `cap`,
    ties first, the rest drawn with a seed.  Only the CHOICE of reads comes from the device; the oracle sees the reads."""
    b, s = top2[:, 0, 2].astype(np.int64), top2[:, 1, 2].astype(np.int64)
    ties = np.where(b == s)[0]
    near = np.where((10 * s >= 9 * b) & (b != s))[0]
    rng = np.random.Generator(np.random.PCG64(seed))
    if near.size > max(0, cap - ties.size):
        near = rng.choice(near, size=max(0, cap - ties.size), replace=False)
    return np.sort(np.concatenate([ties[:cap], near])).astype(np.int64), int(ties.size)


def _sample_check(oracle_mod, genome, cfg, reads, lens, d_top2, top2, nw, idx, nw_cap=None):
    from test_gpu_mapq import check_mapq
    idx = np.unique(idx)
    want = oracle_mod.map_reads_parallel(genome, cfg.frag_len, cfg.overlap, reads[idx], lens[idx], strands=cfg.strands)
    bad = np.where((top2[idx] != want).any(axis=(1, 2)))[0]
    assert bad.size == 0, (bad.size, idx[bad[0]], top2[idx][bad[0]].tolist(), want[bad[0]].tolist())
    # next row f1 on the same sample: device filter on the device records, oracle filter on the oracle's records
    import torch
    check_mapq(oracle_mod, d_top2[torch.from_numpy(idx).to(d_top2.device)].contiguous(), want, f"config {cfg.c}")
    sub = np.arange(idx.size) if nw_cap is None or idx.size <= nw_cap else np.linspace(0, idx.size - 1, nw_cap).astype(np.int64)
    ws, wp, wc, wn = oracle_mod.nw_align(genome, cfg.frag_len, cfg.overlap, reads[idx[sub]], lens[idx[sub]], want[sub], cigar_stride=64)
    score, pos, cigar, ncig = nw
    j = idx[sub]
    assert (score[j] == ws).all() and (pos[j] == wp).all() and (ncig[j] == wn).all()
    for k, i in enumerate(j):
        n = min(int(wn[k]), cigar.shape[1], 64)
        assert (cigar[i, :n] == wc[k, :n]).all(), (i, cigar[i, :n], wc[k, :n])
    return want


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
    return G, top2, top2.cpu().numpy(), (sc.cpu().numpy(), pos.cpu().numpy(), cig.cpu().numpy().view(np.uint32), nc.cpu().numpy()), info


def _truth_rate(cfg, r, top2):
    """Reported, not asserted bit-for-bit: top-1 fragment within +-1 of the true fragment."""
    true_frag = r["start"] // cfg.frag_len
    return float(np.mean(np.abs(top2[:, 0, 0] - true_frag) <= 1))


def test_config2_full_100k_reads(oracle_mod):
    cfg = gen.config(2)
    genome, _ = cfg.genome()
    r = cfg.reads(genome)
    G, d_top2, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"])
    assert top2.shape == (100_000, 2, 4) and G.n_frag == 1124
    assert info["variant"] == 7                                          # the configuration bench.py times: the two-pass scan
    _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 22))
    idx = rng.choice(100_000, size=max(640, 40 * CORES), replace=False)
    rep, n_ties = _repeat_like(top2, 10 * CORES, gen.S0 + 23)
    _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], d_top2, top2, nw, np.concatenate([idx, rep]), nw_cap=256)
    assert rep.size > 0                                                  # the supplement is not vacuous on this workload
    assert _truth_rate(cfg, r, top2) > 0.9                              # sanity of the workload, not parity


def test_config3_length_sweep_geometry(oracle_mod):
    cfg = gen.config(3)
    genome, _ = cfg.genome()
    r = cfg.reads(genome, limit=256)                                    # 15 groups x 256 reads, lengths 36..250 in one call
    G, d_top2, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"], cigar_stride=64)
    _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 32))
    per = max(10, CORES)
    idx = np.concatenate([g * 256 + rng.choice(256, size=per, replace=False) for g in range(15)])
    rep, _ = _repeat_like(top2, 4 * CORES, gen.S0 + 33)                  # short reads: many near-repeats by chance
    _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], d_top2, top2, nw, np.concatenate([idx, rep]), nw_cap=256)


def test_config3_each_length_on_its_own(oracle_mod):
    """bench.py --config 3 --read-len L maps one length per call (its own max_len, hence its own tile and table geometry):
    36 and 51 bp take the short-query path, 250 bp the small pass-1 tile."""
    cfg = gen.config(3)
    genome, _ = cfg.genome()
    for gi, m in ((0, 36), (3, 51), (12, 250)):
        n, mm, rate = cfg.groups[gi]
        assert mm == m
        r = gen.make_reads(genome, 2048, m, cfg.reads_seed + 100 * gi, sub_rate=rate)
        G, d_top2, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"], cigar_stride=64)
        _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
        rng = np.random.Generator(np.random.PCG64(gen.S0 + 34 + gi))
        idx = rng.choice(2048, size=2 * CORES, replace=False)
        rep, _ = _repeat_like(top2, CORES, gen.S0 + 35 + gi)
        _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], d_top2, top2, nw, np.concatenate([idx, rep]), nw_cap=64)


def test_config5_throughput_geometry(oracle_mod):
    cfg = gen.config(5)
    genome, _ = cfg.genome()
    r = cfg.reads(genome, limit=20_000)
    G, d_top2, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"])
    _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 52))
    idx = rng.choice(20_000, size=max(320, 20 * CORES), replace=False)
    rep, _ = _repeat_like(top2, 6 * CORES, gen.S0 + 53)
    _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], d_top2, top2, nw, np.concatenate([idx, rep]), nw_cap=256)


@pytest.mark.skipif(os.environ.get("MSS_SKIP_CHR1") == "1", reason="MSS_SKIP_CHR1=1")
def test_config4_chr1_sized_genome(oracle_mod):
    """249 Mbp with N runs and planted duplicates, F = 16384: the genome no longer fits L2 tiles of one block range.  At
    least half of the compared reads start inside a planted duplicate (source or copy): the other copy is their second
    place, which is what the repeat filter exists for."""
    cfg = gen.config(4)
    genome, info_g = cfg.genome()
    r = cfg.reads(genome, limit=1024)
    G, d_top2, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"], cigar_stride=64)
    assert G.n_frag == 15_198
    _properties(top2, r["lens"], G.n_frag, cfg.frag_len)
    start = r["start"]
    in_dup = np.zeros(start.size, dtype=bool)
    for src, dst, L, _rate in info_g["dups"]:
        in_dup |= ((start >= src) & (start < src + L)) | ((start >= dst) & (start < dst + L))
    n_total = max(32, 2 * CORES)
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 42))
    dup_idx = np.where(in_dup)[0]
    assert dup_idx.size >= n_total // 2, dup_idx.size
    pick_dup = rng.choice(dup_idx, size=n_total // 2, replace=False)
    pick_other = rng.choice(np.where(~in_dup)[0], size=n_total - n_total // 2, replace=False)
    want = _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], d_top2, top2, nw, np.concatenate([pick_dup, pick_other]))
    # the duplicates do exercise second place: most of the reads inside one see a strong second fragment
    strong = 10 * want[:, 1, 2].astype(np.int64) >= 6 * want[:, 0, 2].astype(np.int64)
    assert strong.sum() >= n_total // 4


@pytest.mark.skipif(os.environ.get("MSS_SKIP_BIG") == "1", reason="MSS_SKIP_BIG=1")
def test_genome_beyond_l2_streams_from_hbm(oracle_mod):
    """Next row f4, single-GPU half (Table 8: 76 bp reads, fragment length 4800, a genome of
    Gbp size).  500 Mbp: packed genome + N mask = 187 MB, more than the 126 MB L2, so every pass over the fragments streams
    from HBM; 104,167 fragments; the two-pass bounds are produced with the chunk loop at its default size."""
    import paper_1403_2136_b200 as mss
    n_bases, F, m = 500_000_000, 4800, 76
    genome, _ = gen.make_genome(n_bases, gen.S0 + 60, gc=0.41)
    r = gen.make_reads(genome, 512, m, gen.S0 + 61, sub_rate=0.20)
    cfg = gen.Config(60, "beyond-l2", n_bases, F, -1, 3, gc=0.41, groups=((512, m, 0.20),))
    G, d_top2, top2, nw, info = _run(cfg, genome, r["reads"], r["lens"], cigar_stride=64)
    assert G.n_frag == -(-n_bases // F) and info["variant"] == 7
    assert n_bases * 3 // 8 > 150e6
    _properties(top2, r["lens"], G.n_frag, F)
    rng = np.random.Generator(np.random.PCG64(gen.S0 + 62))
    idx = rng.choice(512, size=max(8, CORES), replace=False)
    rep, _ = _repeat_like(top2, max(2, CORES // 4), gen.S0 + 63)
    _sample_check(oracle_mod, genome, cfg, r["reads"], r["lens"], d_top2, top2, nw, np.concatenate([idx, rep]))
    assert _truth_rate(cfg, r, top2) > 0.3                              # sanity only: 76 bp at 20 % divergence + indels against 1e9 positions
