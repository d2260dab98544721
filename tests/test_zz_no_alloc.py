"""-m gpu, collected last: mss_map_reads_static, the entry point that allocates nothing (the scan's scratch is a static device
array inside the library, include/mss.h).  Its records must equal those of the existing path (mss_map_reads with a caller
workspace) bit for bit -- the bar of every other parity test here -- on two calls in a row that share the array: the second
call maps DIFFERENT reads (another count, another length mix, another strand setting), so whatever the first call left in
the scratch would show.  Also: the records equal the oracle's, the call makes no device allocation, and a batch beyond the
array's size is refused with MSS_ERR_STATIC_LIMIT before anything is launched."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


def _inputs(reads, lens):
    from gpu_util import to_dev
    rp, rn = gen.pack_reads(reads, lens)
    return to_dev(rp), to_dev(rn), to_dev(np.asarray(lens, dtype=np.int32))


def test_static_scratch_entry_point_matches_the_workspace_path(oracle_mod):
    import torch
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome
    mss.mss_set_scan_variant(0)
    mss.mss_set_pass1_geometry(0, 0, -1)
    mss.mss_set_two_pass_chunk_bytes(0)
    cfg = gen.config(1)
    g, _ = cfg.genome()
    r = cfg.reads(g)
    reads, lens = r["reads"].copy(), r["lens"].copy()
    reads[1::2] = np.stack([gen.revcomp(x) for x in reads[1::2]])
    reads[5, 40] = gen.N
    lens[11] = 99; reads[11, 99:] = gen.N
    G = load_genome(g, cfg.frag_len, -1)
    assert mss.mss_static_scratch_bytes() == 32 << 20
    mss.mss_static_init()                                   # set-up: once per device, with the device current
    mss.mss_static_init()                                   # idempotent

    calls = [(reads, lens, 3), (reads[120:170, :60].copy(), np.minimum(lens[120:170], 60).astype(np.int32), 1)]
    for k, (rd, ln, strands) in enumerate(calls):           # two calls in a row on the shared array
        d_reads, d_mask, d_lens = _inputs(rd, ln)
        m = int(rd.shape[1])
        want_dev = mss.mss_map_reads(G, d_reads, d_mask, d_lens, m, mss.Scoring(), strands)       # existing path: caller workspace
        info = mss.mss_get_last_launch()
        out = torch.full((rd.shape[0], 2, 4), -7, dtype=torch.int32, device=d_lens.device)       # the caller's output buffer
        torch.cuda.synchronize()
        n_alloc = torch.cuda.memory_stats()["allocation.all.allocated"]     # allocation requests so far (frees do not count)
        got_dev = mss.mss_map_reads_static(G, d_reads, d_mask, d_lens, m, out, mss.Scoring(), strands)
        torch.cuda.synchronize()
        assert torch.cuda.memory_stats()["allocation.all.allocated"] == n_alloc     # nothing came from torch's allocator either
        assert mss.mss_get_last_launch()["variant"] == info["variant"]                           # the same kernels ran
        got, want = got_dev.cpu().numpy(), want_dev.cpu().numpy()
        assert (got == want).all(), f"call {k}: static-scratch records differ from the workspace path"
        ref = oracle_mod.map_reads_parallel(g, cfg.frag_len, -1, rd, ln, strands=strands)
        assert (got == ref).all(), f"call {k}: records differ from the oracle"

    # again the first batch: the array now holds the second call's bounds
    d_reads, d_mask, d_lens = _inputs(reads, lens)
    out = torch.zeros((reads.shape[0], 2, 4), dtype=torch.int32, device=d_lens.device)
    mss.mss_map_reads_static(G, d_reads, d_mask, d_lens, 100, out, mss.Scoring(), 3)
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == oracle_mod.map_reads_parallel(g, cfg.frag_len, -1, reads, lens, strands=3)).all()


def test_static_scratch_limit_is_enforced():
    import torch
    import paper_1403_2136_b200 as mss
    from gpu_util import load_genome
    g = gen.make_genome(400_000, 91)[0]                     # 400 fragments of 1000: 1.6 kB of bounds per read, both strands
    G = load_genome(g, 1000, -1)
    n = 200_000                                             # far beyond 32 MiB of scratch whatever path is taken
    d_reads = torch.zeros((n, 7), dtype=torch.int32, device="cuda")
    d_lens = torch.full((n,), 100, dtype=torch.int32, device="cuda")
    out = torch.full((n, 2, 4), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(mss.MssError) as e:
        mss.mss_map_reads_static(G, d_reads, None, d_lens, 100, out)
    assert e.value.status == mss.MSS_ERR_STATIC_LIMIT and "static" in str(e.value)
    torch.cuda.synchronize()
    assert (out == -7).all()                                # refused before anything was launched
    # an empty batch is fine, bad arguments are still bad arguments
    mss.mss_map_reads_static(G, d_reads[:0], None, d_lens[:0], 100, out[:0])
    with pytest.raises(mss.MssError) as e:
        mss.mss_map_reads_static(G, d_reads[:4], None, d_lens[:4], 100, out[:4], strands=7)
    assert e.value.status == -1
