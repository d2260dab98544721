"""-m gpu: repeat filter + MAPQ (next row f1) through the C ABI against oracle_mapq_filter.

The device filter runs on the device's own top-2 records, the oracle's filter on the oracle's top-2 records of the same
reads (no oracle input comes from the CUDA path; the records themselves are compared first).  `mapped` must agree exactly
for the default rule and for MAPQ cutoffs; MAPQ is a float32 store of a double, compared at 1e-6 relative."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu

THRESHOLDS = (-1.0, 15.2, 62.0, 0.0, 100.0)
MAPQ_RTOL = 1e-6


def check_mapq(oracle_mod, d_top2, want_top2, ctx=""):
    """d_top2: device records (torch); want_top2: the oracle's records of the same reads (numpy)."""
    import torch
    import paper_1403_2136_b200 as mss
    assert (d_top2.cpu().numpy() == want_top2).all(), f"{ctx}: records differ, MAPQ not comparable"
    for thr in THRESHOLDS:
        mapped, mapq = mss.mss_mapq_filter(d_top2, thr)
        torch.cuda.synchronize()
        wm, wq = oracle_mod.mapq_filter(want_top2, thr)
        got_m, got_q = mapped.cpu().numpy(), mapq.cpu().numpy().astype(np.float64)
        # a cutoff decision is taken in double on both sides; it could differ only if MAPQ sat within an ulp of the cutoff
        undecidable = np.isfinite(wq) & (np.abs(wq - thr) < 1e-9) if thr >= 0 else np.zeros(len(wq), dtype=bool)
        bad = np.where((got_m != wm) & ~undecidable)[0]
        assert bad.size == 0, f"{ctx} thr={thr}: mapped differs at {bad[:5]}: {want_top2[bad[0]].tolist()}"
        inf = np.isinf(wq)
        assert (np.isinf(got_q) == inf).all() and (got_q[inf] > 0).all()
        fin = ~inf
        assert np.allclose(got_q[fin], wq[fin], rtol=MAPQ_RTOL, atol=0.0), f"{ctx}: MAPQ differs"
    return oracle_mod.mapq_filter(want_top2)[0]


def test_mapq_on_tiny_top2(oracle_mod):
    """Every read of config 1 (both strands), plus reads made to hit duplicated blocks (ties and ratios >= .9)."""
    import torch
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, to_dev
    cfg = gen.config(1)
    g, _ = cfg.genome()
    g = g.copy()
    g[31_100:31_400] = g[7_100:7_400]                      # an exact duplicate: reads from it tie (ratio 1)
    dup = g[12_050:12_350].copy()
    dup[::9] = (dup[::9] + 1) % 4                          # an 11 % diverged copy: ratios around .9
    g[40_050:40_350] = dup
    r = cfg.reads(g)
    reads, lens = r["reads"].copy(), r["lens"].copy()
    reads[0] = g[7_150:7_250]; reads[1] = gen.revcomp(g[7_180:7_280]); reads[2] = g[12_100:12_200]; reads[3] = g[12_180:12_280]
    reads[4] = gen.N                                       # all-N read: best score 0 -> unmapped
    lens[:5] = 100
    G = load_genome(g, cfg.frag_len, -1)
    rp, rn = gen.pack_reads(reads, lens)
    top2 = mss.mss_map_reads(G, to_dev(rp), to_dev(rn), to_dev(lens), 100, mss.Scoring(), 3)
    torch.cuda.synchronize()
    want = oracle_mod.map_reads_parallel(g, cfg.frag_len, -1, reads, lens, strands=3)
    mapped = check_mapq(oracle_mod, top2, want, "tiny")
    assert want[0, 0, 2] == want[0, 1, 2] == 500 and mapped[0] == 0 and mapped[1] == 0      # the tie is rejected as a repeat
    assert want[4, 0, 2] == 0 and mapped[4] == 0
    assert 20 < mapped.sum() < 200                         # the workload maps most reads and rejects some


def test_mapq_single_fragment_and_zero_scores(oracle_mod):
    """nfrag = 1: second.frag = -1 is a real output (p = 0, MAPQ = +inf, mapped); a read scoring 0 everywhere is unmapped."""
    import torch
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome, to_dev
    g = gen.make_genome(3000, 61)[0]
    g[g == 0] = 1                                          # no A and no T in the genome: an all-A read scores 0 on
    g[g == 3] = 2                                          # both strands (its reverse complement is all T)
    reads = np.stack([g[500:560], gen.revcomp(g[900:960]), np.zeros(60, dtype=np.uint8)])
    lens = np.full(3, 60, dtype=np.int32)
    G = load_genome(g, 3000, -1)
    rp, rn = gen.pack_reads(reads, lens)
    top2 = mss.mss_map_reads(G, to_dev(rp), to_dev(rn), to_dev(lens), 60, mss.Scoring(), 3)
    torch.cuda.synchronize()
    want = oracle_mod.map_reads(g, 3000, -1, reads, lens, strands=3)
    assert (want[:, 1, 0] == -1).all() and want[2, 0, 2] == 0
    mapped = check_mapq(oracle_mod, top2, want, "one fragment")
    assert mapped.tolist() == [1, 1, 0]


def test_mapq_constructed_records(oracle_mod):
    """Hand-made records on both sides of every boundary: exactly .9, one below / above it, the 62 cutoff (ratio .650 /
    .651), ties, no second fragment, second score 0, best 0, no best; plus a sweep of all (best, second) up to 160."""
    import torch
    recs = [[[3, 1, 100, 0], [5, 2, 89, 0]], [[3, 1, 100, 0], [5, 2, 90, 1]], [[3, 1, 100, 0], [5, 2, 91, 1]],
            [[3, 1, 50, 0], [5, 2, 45, 1]], [[3, 1, 1000, 0], [5, 2, 650, 1]], [[3, 1, 1000, 0], [5, 2, 651, 1]],
            [[3, 1, 100, 0], [-1, 0, 0, 0]], [[3, 1, 100, 0], [9, 0, 0, 0]], [[-1, 0, 0, 0], [-1, 0, 0, 0]],
            [[0, 0, 0, 0], [1, 0, 0, 0]], [[2, 9, 200, 1], [7, 0, 200, 0]], [[2, 9, 32767, 1], [7, 0, 1, 0]],
            [[2, 9, 32767, 1], [7, 0, 32766, 0]], [[2, 9, 1, 0], [7, 0, 1, 0]], [[2, 9, 1, 0], [7, 0, 0, 0]]]
    for b in range(0, 161):
        for s in range(0, b + 1):
            recs.append([[1, 0, b, 0], [4, 0, s, 1]])
    want = np.array(recs, dtype=np.int32)
    d = torch.from_numpy(want).cuda()
    mapped = check_mapq(oracle_mod, d, want, "constructed")
    assert mapped[:4].tolist() == [1, 0, 0, 0]             # below .9 only
    import paper_1403_2136_b200 as mss
    m62, _ = mss.mss_mapq_filter(d, 62.0)
    assert m62.cpu().numpy()[[4, 5]].tolist() == [1, 0]
    mdef, _ = mss.mss_mapq_filter(d)                       # the binding's default is the paper's exact rule
    assert (mdef.cpu().numpy() == mapped).all()
