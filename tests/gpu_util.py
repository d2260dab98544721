"""Helpers for the -m gpu parity tests: marshal gen/ inputs to the device and call the C ABI through the binding."""
import numpy as np

import gen


def to_dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a).view(np.int32) if a.dtype == np.uint32 else np.ascontiguousarray(a))
    return t.cuda()


def load_genome(codes, frag_len, overlap):
    import paper_1403_2136_b200 as mss
    packed, nmask = gen.pack_2bit(codes)
    return mss.mss_genome_load(to_dev(packed), to_dev(nmask), int(codes.size), frag_len, overlap)


def map_reads(g, reads, lens, strands=3, match=5, mismatch=-4, variant=0, with_mask=True, stride_words=None):
    import torch
    import paper_1403_2136_b200 as mss
    reads = np.asarray(reads, dtype=np.uint8)
    lens = np.asarray(lens, dtype=np.int32)
    rp, rn = gen.pack_reads(reads, lens, stride_words)
    mss.mss_set_scan_variant(variant)
    try:
        out = mss.mss_map_reads(g, to_dev(rp), to_dev(rn) if with_mask else None, to_dev(lens), int(reads.shape[1]),
                                mss.Scoring(match, mismatch, -26), strands)
        torch.cuda.synchronize()
    finally:
        mss.mss_set_scan_variant(0)
    return out.cpu().numpy()


def nw_align(g, reads, lens, top2, match=5, mismatch=-4, gap=-26, pad=30, cigar_stride=None):
    import torch
    import paper_1403_2136_b200 as mss
    reads = np.asarray(reads, dtype=np.uint8)
    lens = np.asarray(lens, dtype=np.int32)
    rp, rn = gen.pack_reads(reads, lens)
    sc, pos, cig, nc = mss.mss_nw_align(g, to_dev(rp), to_dev(rn), to_dev(lens), int(reads.shape[1]),
                                        to_dev(np.ascontiguousarray(top2, dtype=np.int32)),
                                        mss.Scoring(match, mismatch, gap), pad, cigar_stride)
    torch.cuda.synchronize()
    return sc.cpu().numpy(), pos.cpu().numpy(), cig.cpu().numpy().view(np.uint32), nc.cpu().numpy()


def map_reads_fast(g, reads, lens, strands=3, match=5, mismatch=-4, variant=0):
    import torch
    import paper_1403_2136_b200 as mss
    reads = np.asarray(reads, dtype=np.uint8)
    lens = np.asarray(lens, dtype=np.int32)
    rp, rn = gen.pack_reads(reads, lens)
    mss.mss_set_scan_variant(variant)
    try:
        out = mss.mss_map_reads_fast(g, to_dev(rp), to_dev(rn), to_dev(lens), int(reads.shape[1]),
                                     mss.Scoring(match, mismatch, -26), strands)
        torch.cuda.synchronize()
    finally:
        mss.mss_set_scan_variant(0)
    return out.cpu().numpy()


def pssm_tables(quals, lens, match=5, mismatch=-4, scale=16):
    """-> (device packed table from mss_pssm_build, its unpacked (pmatch, pmismatch) int32 host copies)."""
    import torch
    import paper_1403_2136_b200 as mss
    d = mss.mss_pssm_build(to_dev(np.ascontiguousarray(quals, dtype=np.uint8)), to_dev(np.asarray(lens, dtype=np.int32)),
                           mss.Scoring(match, mismatch, -26), scale)
    torch.cuda.synchronize()
    h = d.cpu().numpy().view(np.uint32)
    pm = (h & 0xFFFF).astype(np.uint16).view(np.int16).astype(np.int32)
    pmm = (h >> 16).astype(np.uint16).view(np.int16).astype(np.int32)
    return d, pm, pmm


def map_reads_pssm(g, reads, lens, d_pssm, strands=3, match=5, mismatch=-4, scale=16, variant=0, bound=None):
    import torch
    import paper_1403_2136_b200 as mss
    reads = np.asarray(reads, dtype=np.uint8)
    lens = np.asarray(lens, dtype=np.int32)
    rp, rn = gen.pack_reads(reads, lens)
    mss.mss_set_scan_variant(variant)
    try:
        out = mss.mss_map_reads_pssm(g, to_dev(rp), to_dev(rn), to_dev(lens), int(reads.shape[1]), d_pssm,
                                     bound or mss.pssm_bound(mss.Scoring(match, mismatch, -26), scale), strands)
        torch.cuda.synchronize()
    finally:
        mss.mss_set_scan_variant(0)
    return out.cpu().numpy()


def nw_align_pssm(g, reads, lens, top2, d_pssm, match=5, mismatch=-4, gap=-26, scale=16, pad=30, cigar_stride=None):
    import torch
    import paper_1403_2136_b200 as mss
    reads = np.asarray(reads, dtype=np.uint8)
    lens = np.asarray(lens, dtype=np.int32)
    rp, rn = gen.pack_reads(reads, lens)
    sc, pos, cig, nc = mss.mss_nw_align_pssm(g, to_dev(rp), to_dev(rn), to_dev(lens), int(reads.shape[1]),
                                             to_dev(np.ascontiguousarray(top2, dtype=np.int32)), d_pssm,
                                             mss.pssm_bound(mss.Scoring(match, mismatch, gap), scale), pad, cigar_stride)
    torch.cuda.synchronize()
    return sc.cpu().numpy(), pos.cpu().numpy(), cig.cpu().numpy().view(np.uint32), nc.cpu().numpy()
