#!/usr/bin/env python
"""Full-coverage parity run (not a pytest: it needs a B200 and, for the large configs, an hour of host cores).

    python tests/full_parity.py --config 2 [--reads N] [--mode plain|fast|pssm] [--out gpurun_out/parity_c2.json]

Maps the config's reads (all of them, or the first N of every group) through the C ABI on cuda:0, then through the CPU
oracle on every host core (one single-threaded oracle process per core, chunk by chunk so progress is visible), and
compares EVERY record bit for bit: top-2 (fragment, window start, score, strand) and the second stage's score, position
and CIGAR.  Writes one JSON summary.  SURVEY.md 8(d) "Oracle timing and coverage": configs 1 and 2 on every read.
The committed summaries of the runs made for a round live under profiles/.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import gen  # noqa: E402
import oracle  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--reads", type=int, default=None, help="first N reads of every group (default: all)")
    ap.add_argument("--mode", default="plain", choices=["plain", "fast", "pssm"])
    ap.add_argument("--read-len", type=int, default=None,
                    help="keep only the reads of this length (config 3: one length of the sweep per call, as bench.py --read-len does)")
    ap.add_argument("--nw-reads", type=int, default=4096, help="reads whose second stage is also compared (evenly spaced)")
    ap.add_argument("--skip", type=int, default=0, help="compare only reads [skip, n) with the oracle (the GPU still maps all)")
    ap.add_argument("--stop", type=int, default=None, help="compare only reads [skip, stop) (one gpurun call lasts at most an hour)")
    ap.add_argument("--variant", type=int, default=0, help="scan variant (0 = automatic, 7 = two-pass)")
    ap.add_argument("--chunk", type=int, default=2048)
    ap.add_argument("--workers", type=int, default=None,
                    help="oracle processes (default: every host core; each holds its own copy of the genome, so use few for Gbp genomes)")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()

    import torch
    import paper_1403_2136_b200 as mss
    cfg = gen.config(args.config)
    genome, _ = cfg.genome()
    r = cfg.reads(genome, limit=args.reads)
    reads, lens = r["reads"], r["lens"]
    if args.read_len is not None:
        keep = lens == args.read_len
        reads, lens = np.ascontiguousarray(reads[keep][:, :args.read_len]), np.ascontiguousarray(lens[keep])
        r = {k: (v[keep] if hasattr(v, "shape") and v.shape[:1] == keep.shape else v) for k, v in r.items()}
        if lens.size == 0:
            raise SystemExit(f"config {cfg.c} has no reads of length {args.read_len}")
    n, m = reads.shape
    dev = torch.device("cuda", 0)
    packed, nmask = gen.pack_2bit(genome)
    rp, rn = gen.pack_reads(reads, lens)
    G = mss.mss_genome_load(torch.from_numpy(packed.view(np.int32)).to(dev), torch.from_numpy(nmask.view(np.int32)).to(dev),
                            int(genome.size), cfg.frag_len, cfg.overlap)
    d_reads, d_mask, d_lens = (torch.from_numpy(rp.view(np.int32)).to(dev), torch.from_numpy(rn.view(np.int32)).to(dev),
                               torch.from_numpy(lens).to(dev))
    sc = mss.Scoring()
    mss.mss_set_scan_variant(args.variant)
    scale = 16
    pm = pmm = None
    t0 = time.perf_counter()
    if args.mode == "fast":
        top2 = mss.mss_map_reads_fast(G, d_reads, d_mask, d_lens, m, sc, cfg.strands)
    elif args.mode == "pssm":
        quals = gen.make_quals(n, m, cfg.reads_seed + 5)
        d_pssm = mss.mss_pssm_build(torch.from_numpy(quals).to(dev), d_lens, sc, scale)
        top2 = mss.mss_map_reads_pssm(G, d_reads, d_mask, d_lens, m, d_pssm, mss.pssm_bound(sc, scale), cfg.strands)
        pm, pmm = oracle.pssm_from_phred(quals, sc.match, sc.mismatch, scale)
    else:
        top2 = mss.mss_map_reads(G, d_reads, d_mask, d_lens, m, sc, cfg.strands)
    if args.mode == "pssm":
        nw = mss.mss_nw_align_pssm(G, d_reads, d_mask, d_lens, m, top2, d_pssm, mss.pssm_bound(sc, scale), 30, 64)
    else:
        nw = mss.mss_nw_align(G, d_reads, d_mask, d_lens, m, top2, sc, 30, 64)
    torch.cuda.synchronize()
    gpu_s = time.perf_counter() - t0
    got = top2.cpu().numpy()
    g_score, g_pos, g_cig, g_nc = (nw[0].cpu().numpy(), nw[1].cpu().numpy(), nw[2].cpu().numpy().view(np.uint32),
                                   nw[3].cpu().numpy())
    info = mss.mss_get_last_launch()

    cores = args.workers or os.cpu_count() or 1
    bad_top2, checked = [], 0
    t0 = time.perf_counter()
    want_all = np.zeros_like(got)
    stop = n if args.stop is None else min(n, args.stop)
    for a in range(args.skip, stop, args.chunk):
        b = min(stop, a + args.chunk)
        if args.mode == "pssm":
            want = oracle.map_reads_pssm_parallel(genome, cfg.frag_len, cfg.overlap, reads[a:b], lens[a:b], pm[a:b], pmm[a:b],
                                                  strands=cfg.strands, workers=cores)
        else:
            want = oracle.map_reads_parallel(genome, cfg.frag_len, cfg.overlap, reads[a:b], lens[a:b], strands=cfg.strands,
                                             workers=cores, fast=(args.mode == "fast"))
        want_all[a:b] = want
        diff = np.where((got[a:b] != want).any(axis=(1, 2)))[0]
        bad_top2 += [int(a + i) for i in diff]
        checked = b
        el = time.perf_counter() - t0
        print(f"[full_parity] {checked}/{n} reads, {len(bad_top2)} differ, {el:.0f} s", file=sys.stderr, flush=True)
    cpu_s = time.perf_counter() - t0

    # second stage on an evenly spaced subset (the oracle's full-matrix NW is the slow part there)
    idx = np.unique(np.linspace(args.skip, stop - 1, min(stop - args.skip, args.nw_reads)).astype(np.int64))
    if args.mode == "pssm":
        ws, wp, wc, wn = oracle.nw_align_pssm(genome, cfg.frag_len, cfg.overlap, reads[idx], lens[idx], want_all[idx], pm[idx],
                                              pmm[idx], scale * sc.gap, cigar_stride=64)
    else:
        ws, wp, wc, wn = oracle.nw_align(genome, cfg.frag_len, cfg.overlap, reads[idx], lens[idx], want_all[idx], cigar_stride=64)
    bad_nw = []
    for k, i in enumerate(idx):
        ok = g_score[i] == ws[k] and g_pos[i] == wp[k] and g_nc[i] == wn[k]
        nc = min(int(wn[k]), 64)
        ok = ok and bool((g_cig[i, :nc] == wc[k, :nc]).all())
        if not ok:
            bad_nw.append(int(i))
    # the NW comparison assumes the GPU hit equals the oracle's hit, which the top-2 comparison establishes
    per_frag = G.n_frag * cfg.frag_len * (2 if cfg.strands == 3 else 1)
    scored = lens if args.mode != "fast" else -(-lens // 2)
    cells = float(np.sum(scored)) * per_frag                               # cells of the whole batch (what the GPU mapped)
    cells_compared = float(np.sum(scored[args.skip:stop])) * per_frag      # cells of the slice the oracle re-computed
    summary = {
        "config": cfg.c, "name": cfg.name, "mode": args.mode, "read_len_filter": args.read_len, "reads": int(n), "read_len_max": int(m), "n_frag": int(G.n_frag),
        "cells": cells, "top2_compared": int(checked - args.skip), "first_read_compared": int(args.skip), "top2_mismatches": len(bad_top2), "first_bad_top2": bad_top2[:5],
        "nw_compared": int(len(idx)), "nw_mismatches": len(bad_nw), "first_bad_nw": bad_nw[:5],
        "ties_best_eq_second": int(np.sum(got[:, 0, 2] == got[:, 1, 2])),
        "ratio_ge_0.9": int(np.sum(10 * got[:, 1, 2].astype(np.int64) >= 9 * got[:, 0, 2].astype(np.int64))),
        "top1_within_1_of_truth": float(np.mean(np.abs(got[:, 0, 0] - r["start"] // cfg.frag_len) <= 1)),
        "gpu_wall_s": gpu_s, "oracle_wall_s": cpu_s, "oracle_cores": cores, "cells_compared": cells_compared,
        "oracle_gcups": cells_compared / cpu_s / 1e9,
        "launch": info, "inputs_sha256": gen.sha256_of(genome, reads, lens),
    }
    line = json.dumps(summary)
    print(line)
    if args.out:
        with open(args.out, "w") as f:
            f.write(line + "\n")
    sys.exit(0 if not bad_top2 and not bad_nw else 1)


if __name__ == "__main__":
    main()
