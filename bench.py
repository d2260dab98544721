#!/usr/bin/env python
"""bench.py -- MaxSS GCUPS of the whole hot path (scan + top-2 + NW) on synthetic config-2 input.

    python bench.py --gpus N --steps K --warmup W            # our CUDA path (C ABI -> libmss.so)
    python bench.py --impl reference ...                     # the CPU oracle as it stands, on the host cores

A step = one pass of every hot-path stage (read prep, tile staging, Kadane scan, fragment max,
top-2, emit, NW) over one batch of reads of BASELINE.json's E. coli-sized config (configs[1]); the genome load (a0,
"once") is timed separately.  One JSON line on stdout (rank 0).  DESIGN.md section 7 explains every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import gen  # noqa: E402

ALGO_INSTR_PER_CELL = 0.75          # one-pass scan: 1 add-max-relu per 2 cells + 1 three-input max per 4 cells
ALGO_INSTR_PER_CELL_PASS1 = 0.375   # two-pass scan, pass 1: 1 add-max-relu per 4 cells + 1 three-input max per 8 cells
ALU_LANES_PER_CLK_SM = 64           # integer/DPX pipe: 16 lanes/clk per SM sub-partition x 4 (guide + measured)
ISSUE_LANES_PER_CLK_SM = 128        # one warp instruction per clock per SM sub-partition
SMEM_BYTES_PER_CLK_SM = 128         # shared-memory data pipe: one 128-byte wavefront per clock per SM
# ncu --set full captures of the dominant kernels at ONE launch size (config 2, 4096 reads); quoted only for that launch
NCU_CAPTURES = {
    "scan_filter_lq_kernel": {"dram_bytes": 2_115_840, "instr_per_cell": 0.814, "smem_bytes_per_cell": 0.5,
                              "source": "profiles/r2_scan_filter_lq_full.md"},
    "scan_filter_lq_kernel_pssm": {"dram_bytes": 3_751_424, "instr_per_cell": 1.044, "smem_bytes_per_cell": 1.0,
                                   "source": "profiles/r2_other_kernels.md"},
    "scan_filter_kernel": {"dram_bytes": 2_019_072, "instr_per_cell": 0.871, "smem_bytes_per_cell": 1.0,
                           "source": "profiles/r1_scan_filter_full.md"},
    "scan_dpx_kernel": {"dram_bytes": 2_043_648, "instr_per_cell": 1.54, "smem_bytes_per_cell": 2.0,
                        "source": "profiles/r1_scan_dpx_full.md"},
}


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        except Exception:
            pass

    def stop(self) -> dict:
        if self.proc:
            self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p))
    return {}


def cpu_baseline(cfg, genome, reads, lens, target_s: float = 15.0) -> dict:
    """The oracle as it stands, on the host cores, on a bounded seeded sample of the same reads."""
    import oracle
    oracle.build()
    cores = os.cpu_count() or 1
    per_read_cells = cfg.cells() / cfg.n_reads
    guess = 1.4e9                                    # cells/s/core of the plain -O3 build (measured in DESIGN.md)
    if per_read_cells / guess > 4 * target_s:          # one read alone would run for minutes (Gbp-sized genomes): not a bounded sample
        return {"value": None, "unit": "GCUPS", "cores": 0, "kind": "oracle",
                "sample": "skipped: one read of this config costs the oracle more than a minute per core"}
    per_core = max(1, int(target_s * guess / per_read_cells))
    n = min(reads.shape[0], cores * per_core)
    t0 = time.perf_counter()
    oracle.map_reads_parallel(genome, cfg.frag_len, cfg.overlap, reads[:n], lens[:n], strands=cfg.strands, workers=cores)
    dt = time.perf_counter() - t0
    cells = per_read_cells * n
    return {"value": cells / dt / 1e9, "unit": "GCUPS", "cores": min(cores, n), "kind": "oracle",
            "sample": f"first {n} reads of the step's batch, all {-(-cfg.genome_len // cfg.frag_len)} fragments, both strands, "
                      f"oracle/maxss_oracle.c -O3 single-threaded per process, {dt:.1f} s wall",
            "reads_per_s": n / dt}


def run_reference(args, cfg):
    """--impl reference: the CPU oracle timed on this arm's config/metric (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    genome, _ = cfg.genome()
    cores = os.cpu_count() or 1
    n = cores * args.ref_reads_per_core
    r = gen.make_reads(genome, n, cfg.groups[0][1], cfg.reads_seed, sub_rate=cfg.groups[0][2])
    per_read_cells = cfg.cells() / cfg.n_reads
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        top2 = oracle.map_reads_parallel(genome, cfg.frag_len, cfg.overlap, r["reads"], r["lens"], strands=cfg.strands,
                                         workers=cores)
        oracle.nw_align(genome, cfg.frag_len, cfg.overlap, r["reads"][:cores], r["lens"][:cores], top2[:cores])
        dt = time.perf_counter() - t0
        if it >= args.warmup:
            times.append(dt)
    ms = 1e3 * sum(times) / len(times)
    val = per_read_cells * n / (ms * 1e-3) / 1e9
    sample = (f"each step: {n} seeded reads of the config ({args.ref_reads_per_core} per core) through the oracle's MaxSS "
              f"stage on all fragments and both strands, plus its NW on {cores} of them")
    line = {"impl": "reference", "metric": "MaxSS GCUPS (scan+top-2+NW step)", "value": val, "unit": "GCUPS", "n_gpus": 0,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": f"config {cfg.c} ({cfg.name}) bounded sample", "reads_per_step": n, "read_len": cfg.groups[0][1],
                       "genome_bp": cfg.genome_len, "frag_len": cfg.frag_len, "overlap": cfg.overlap, "strands": "both"},
            "cpu_baseline": {"value": val, "unit": "GCUPS", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "GCUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "reads_per_s": n / (ms * 1e-3)}
    print(json.dumps(line), flush=True)


def free_port() -> int:
    import socket
    sk = socket.socket()
    sk.bind(("127.0.0.1", 0))
    port = sk.getsockname()[1]
    sk.close()
    return port


def respawn_under_torchrun(args) -> None:
    """`python bench.py --gpus N` (N > 1) with no launcher around it: start the N ranks ourselves, exactly as the driver
    would (one process per GPU, torch.distributed.run, rendezvous on 127.0.0.1), and hand back their exit code."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def rank_inputs(cfg, args, rank: int, world: int, genome):
    """This rank's batch of reads: the config's own reads on one GPU; with several ranks (weak scaling) or with --reads /
    --read-len every rank draws its own batch from the same recipe, the seed offset by the rank."""
    groups = [g for g in cfg.groups if args.read_len in (None, g[1])]
    if not groups:
        raise SystemExit(f"config {cfg.c} has no read group of length {args.read_len}")
    m = max(g[1] for g in groups)
    n_reads = args.reads or sum(g[0] for g in groups)
    r = None
    if args.reads is None and args.read_len is None and world == 1:
        r = cfg.reads(genome)
    if r is None:
        outs = []
        per = max(1, n_reads // len(groups))
        for gi, (_, mm, rate) in enumerate(groups):
            o = gen.make_reads(genome, per, mm, cfg.reads_seed + 100 * gi + 7919 * rank, sub_rate=rate,
                               indel_prob=cfg.indel_prob, both_strands=cfg.both_strands, avoid_n=cfg.avoid_n)
            if mm < m:
                pad = np.full((per, m), gen.N, dtype=np.uint8); pad[:, :mm] = o["reads"]; o["reads"] = pad
            outs.append(o)
        r = {k: np.concatenate([o[k] for o in outs]) for k in outs[0]}
    reads, lens = r["reads"].copy(), r["lens"]
    n_with_n = 0
    if args.n_frac > 0:                # real reads carry N calls (the profile has an N row): one N in a fraction of the reads
        rng = np.random.Generator(np.random.PCG64(cfg.reads_seed + 31 + 7919 * rank))
        pick = np.where(rng.random(reads.shape[0]) < args.n_frac)[0]
        reads[pick, rng.integers(0, np.maximum(lens[pick], 1))] = gen.N
        n_with_n = int(pick.size)
    return reads, lens, m, n_with_n


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5; 6 = whole-genome-sized); the metric is quoted on 2")
    ap.add_argument("--reads", type=int, default=None, help="reads per step per GPU (default: the config's own count)")
    ap.add_argument("--variant", type=int, default=0, help="scan kernel variant (0 = automatic)")
    ap.add_argument("--read-len", type=int, default=None,
                    help="diagnostic: keep only the config's read groups of this length (config 3's sweep, one length at a time)")
    ap.add_argument("--mode", default="plain", choices=["plain", "fast", "pssm"],
                    help="diagnostic: time the next-row scans (MaxSSmap_fast / base-quality PSSM) instead of the plain scan")
    ap.add_argument("--n-frac", type=float, default=0.0, help="diagnostic: fraction of reads that get one N (they take the unfiltered path)")
    ap.add_argument("--query-sets", type=int, default=0, help="pass 1: 32-query sets per block (1, 2, 4; 0 = default) -- config 5's reads-per-block sweep")
    ap.add_argument("--tile", type=int, default=0, help="pass 1: window starts per tile (0 = automatic)")
    ap.add_argument("--arith", type=int, default=-1, help="pass 1 arithmetic: 0 int16 DPX, 1 fp16, 2 e5m2 bytes, -1 automatic")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-nw", action="store_true", help="time the MaxSS stage only (diagnostic; not a bench value)")
    ap.add_argument("--ref-reads-per-core", type=int, default=2)
    ap.add_argument("--cigar-stride", type=int, default=16)
    ap.add_argument("--plumbing-only", action="store_true",
                    help="test hook: run the launch / sharding / max-over-ranks / rank-0-print path on the CPU (gloo) with the "
                         "device work replaced by a sleep; prints no metric value")
    args = ap.parse_args()
    cfg = gen.config(args.config)
    if args.impl == "reference":
        run_reference(args, cfg)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        respawn_under_torchrun(args)

    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != max(1, args.gpus) and rank == 0:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} but the launcher started {world} rank(s); reporting n_gpus={world}\n")

    if args.plumbing_only:
        plumbing_only(args, cfg, rank, world)
        return

    import paper_1403_2136_b200 as mss
    if not os.path.exists(mss.lib_path()) and local == 0:
        from paper_1403_2136_b200 import build as mss_build      # in-tree build of libmss.so (nvcc, sm_100a); no fallback exists
        mss_build.build()
    for _ in range(600):                                         # other local ranks wait for rank 0's build
        if os.path.exists(mss.lib_path()):
            break
        time.sleep(0.5)

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    from paper_1403_2136_b200.shard import max_over_ranks

    # ---- inputs: genome replicated, reads sharded by rank (independent units, no data-path collective) ------------
    genome, _ = cfg.genome()
    reads, lens, m, n_with_n = rank_inputs(cfg, args, rank, world, genome)
    n_reads = reads.shape[0]
    packed, nmask = gen.pack_2bit(genome)
    rp, rn = gen.pack_reads(reads, lens)
    h_reads = torch.from_numpy(rp.view(np.int32)).pin_memory()
    h_mask = torch.from_numpy(rn.view(np.int32)).pin_memory()
    h_lens = torch.from_numpy(lens).pin_memory()

    t0 = time.perf_counter()
    d_packed = torch.from_numpy(packed.view(np.int32)).to(dev)
    d_nmask = torch.from_numpy(nmask.view(np.int32)).to(dev)
    G = mss.mss_genome_load(d_packed, d_nmask, int(genome.size), cfg.frag_len, cfg.overlap)
    torch.cuda.synchronize()
    genome_load_ms = 1e3 * (time.perf_counter() - t0)

    d_reads, d_mask, d_lens = h_reads.to(dev), h_mask.to(dev), h_lens.to(dev)
    sc = mss.Scoring()
    mss.mss_set_scan_variant(args.variant)
    mss.mss_set_pass1_geometry(args.query_sets, args.tile, args.arith)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)          # > 126 MB L2
    stream = torch.cuda.current_stream()
    scored = lens.astype(np.float64) if args.mode != "fast" else np.ceil(lens.astype(np.float64) / 2)   # fast: every other base
    ns = 2 if cfg.strands == 3 else 1
    cells_step = float(np.sum(scored)) * G.n_frag * cfg.frag_len * ns
    d_qual, pssm_scale = None, 16
    if args.mode == "pssm":
        d_qual = torch.from_numpy(gen.make_quals(n_reads, m, cfg.reads_seed + 5)).to(dev)

    def step():
        """resident inputs -> top-2 records -> NW score/pos/CIGAR, all on the device; returns the event triple."""
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(stream)
        if args.mode == "fast":
            top2 = mss.mss_map_reads_fast(G, d_reads, d_mask, d_lens, m, sc, cfg.strands)
        elif args.mode == "pssm":
            d_pssm = mss.mss_pssm_build(d_qual, d_lens, sc, pssm_scale)
            bound = mss.pssm_bound(sc, pssm_scale)
            top2 = mss.mss_map_reads_pssm(G, d_reads, d_mask, d_lens, m, d_pssm, bound, cfg.strands)
        else:
            top2 = mss.mss_map_reads(G, d_reads, d_mask, d_lens, m, sc, cfg.strands)
        e1.record(stream)
        if not args.no_nw:
            if args.mode == "pssm":
                mss.mss_nw_align_pssm(G, d_reads, d_mask, d_lens, m, top2, d_pssm, bound, 30, args.cigar_stride)
            else:
                mss.mss_nw_align(G, d_reads, d_mask, d_lens, m, top2, sc, 30, args.cigar_stride)
        e2.record(stream)
        return e0, e1, e2, top2

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        flush.fill_(1)
        step()
    launch_info = mss.mss_get_last_launch()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    evs = []
    barrier()
    mss.mss_set_pass_timing(True)
    pass_ms = []
    for _ in range(args.steps):
        flush.fill_(1)                     # L2 flush between timed iterations (inputs are smaller than L2)
        a, b, c, top2 = step()
        evs.append((a, b, c))
        pass_ms.append(mss.mss_get_pass_times())       # waits for this step's scan only (two-pass path; else (0, 0))
    barrier()
    mss.mss_set_pass_timing(False)
    scan_ms = [a.elapsed_time(b) for a, b, _ in evs]
    nw_ms = [b.elapsed_time(c) for _, b, c in evs]
    step_ms = [a.elapsed_time(c) for a, _, c in evs]
    own_ms = sum(step_ms)                   # device time of exactly K steps (the flush writes are outside the events)
    clocks = sampler.stop()
    total_ms = max_over_ranks(own_ms, dev)
    ms_per_step = total_ms / args.steps

    # ---- e2e: host buffers through the C ABI, copies inside the timed region ----------------------------------------
    e2e = None
    if args.mode == "plain":
        out = mss.mss_map_align_host(G, h_reads, h_mask, h_lens, m, sc, cfg.strands, 30, args.cigar_stride)   # warm-up
        e2e_times = []
        for _ in range(max(1, min(args.steps, 2))):
            flush.fill_(1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            out = mss.mss_map_align_host(G, h_reads, h_mask, h_lens, m, sc, cfg.strands, 30, args.cigar_stride, out=out)
            e2e_times.append(time.perf_counter() - t0)
        e2e_s = max_over_ranks(sum(e2e_times) / len(e2e_times), dev)
        h2d = h_reads.numel() * 4 + h_mask.numel() * 4 + h_lens.numel() * 4
        d2h = sum(v.numel() * v.element_size() for v in out.values())
        same = bool((out["top2"] == top2.cpu()).all())
        e2e = {"value": cells_step * world / e2e_s / 1e9, "unit": "GCUPS", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * e2e_s, "matches_device_path": same,
               "api": "mss_map_align_host (pinned host buffers in/out)"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peaks = measured_peaks()
    sm_max = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    clk = sm_max * 1e6
    peak_instr = n_sm * ALU_LANES_PER_CLK_SM * clk                        # thread-instr/s, ALU/DPX pipe at max clock
    scan_avg_ms = sum(scan_ms) / len(scan_ms)
    probe_rate, _ = mss.mss_probe_dpx_peak(2048)
    peak_source = f"{n_sm} SMs x {ALU_LANES_PER_CLK_SM} lanes/clk x {sm_max:.0f} MHz (clocks.max.sm of MEASURED_PEAKS.json)"
    p1_ms = sum(a for a, _ in pass_ms) / len(pass_ms)
    p2_ms = sum(b for _, b in pass_ms) / len(pass_ms)
    two_pass = launch_info["variant"] == 7 and p1_ms > 0
    genome_bytes = cfg.genome_len * 3 / 8                                   # 2-bit words + N mask
    l2_resident = genome_bytes < 100e6
    n_chunks = max(1, launch_info["launches"] // 2) if two_pass else 1
    if two_pass:
        # the dominant kernel is pass 1, which touches every cell of the step
        kernel = "scan_filter_lq_kernel" if launch_info["pass1_kernel"] >= 2 else "scan_filter_kernel"
        kname = f"{kernel} (pass 1 of the two-pass scan)"
        kernel_ms, algo = p1_ms, ALGO_INSTR_PER_CELL_PASS1
        # DRAM bytes the launch has to move: the genome once per chunk of reads while it fits L2 (else once per resident wave
        # of blocks: not modelled, null), the reads once, the 16-bit bounds written by pass 1 (and read back by pass 2)
        bounds_bytes = n_reads * ns * G.n_frag * 2
        traffic_model = (genome_bytes * n_chunks + h_reads.numel() * 4 + bounds_bytes) if l2_resident else None
    else:
        kernel = "scan_dpx_kernel"
        kname, kernel_ms, algo = kernel, scan_avg_ms, ALGO_INSTR_PER_CELL
        traffic_model = (genome_bytes + h_reads.numel() * 4) if l2_resident else None
    cap = NCU_CAPTURES[kernel + ("_pssm" if two_pass and launch_info["pass1_kernel"] == 5 else "")]
    cells_per_clk_sm = cells_step / (kernel_ms * 1e-3) / n_sm / clk
    achieved = cells_step * algo / (kernel_ms * 1e-3)
    same_launch_as_capture = (args.config == 2 and n_reads == 4096 and args.mode in ("plain", "pssm") and m == 100 and args.n_frac == 0)
    roofline = {
        "bound": "alu", "kernel": kname, "achieved": achieved / 1e12, "peak": peak_instr / 1e12, "unit": "T thread-instr/s",
        "frac": achieved / peak_instr,
        # ncu DRAM bytes are quoted only for the launch that was captured (config 2, 4096 reads); other launches get the model
        "traffic": cap["dram_bytes"] if same_launch_as_capture else None, "traffic_source": cap["source"],
        "traffic_model_bytes": traffic_model,
        "traffic_model": "genome (2-bit + N mask) once per chunk of reads + packed reads + 16-bit pass-1 bounds; the genome stays in L2"
                         if l2_resident else "genome larger than L2: streamed from HBM once per wave of blocks, not modelled",
        "peak_source": peak_source, "algorithmic_instr_per_cell": algo, "cells_per_launch": cells_step / n_chunks,
        "launches_per_step": n_chunks, "kernel_ms": kernel_ms, "pass2_ms": p2_ms if two_pass else None,
        "kernel_share_of_step": kernel_ms / (sum(step_ms) / len(step_ms)),
        "cells_per_clk_sm": cells_per_clk_sm,
        "probe_dpx_peak": probe_rate / 1e12, "frac_of_probe": achieved / probe_rate if probe_rate > 0 else None,
        # SURVEY 8(d) fraction (B): the whole scan against the exact one-pass floor of 0.75 instr/cell (may exceed 1: pass 1
        # composes two Kadane steps per instruction and pass 2 restores exactness on ~1 % of the fragments)
        "frac_survey_B": cells_step * ALGO_INSTR_PER_CELL / (scan_avg_ms * 1e-3) / peak_instr,
        # what actually limits the kernel (ncu, profiles/): instructions issued per cell against one warp instruction per
        # clock per sub-partition, and operand bytes per cell against the 128 B/clk/SM shared-memory pipe
        "issue_frac": cells_per_clk_sm * cap["instr_per_cell"] / ISSUE_LANES_PER_CLK_SM,
        "smem_frac": cells_per_clk_sm * cap["smem_bytes_per_cell"] / SMEM_BYTES_PER_CLK_SM,
        "instr_per_cell_profiled": cap["instr_per_cell"], "smem_bytes_per_cell": cap["smem_bytes_per_cell"],
        "limiter": ("ALU pipe (PRMT operand selection, DPX add-max and 3-input max: 96 % busy)" if cap is NCU_CAPTURES["scan_filter_lq_kernel_pssm"]
                    else "issue slots + ALU pipe (PRMT widening and the 3-input max); shared memory at about half its rate"
                    if kernel == "scan_filter_lq_kernel" else "shared-memory wavefronts"),
        "limiter_source": cap["source"],
        "note": ("frac counts the algorithmic 0.375 instr/cell against the ALU/DPX pipe alone (BASELINE.json's metric); this kernel issues "
                 "the add-max-relu as HFMA2.RELU on the FMA pipe and only the 3-input max on the ALU pipe, so the bound that holds is "
                 "issue_frac (all issued instructions against one warp instruction per clock per sub-partition)")
                if kernel == "scan_filter_lq_kernel" else None,
    }
    line = {
        "metric": "MaxSS GCUPS (scan+top-2+NW step)", "value": cells_step * world / (ms_per_step * 1e-3) / 1e9,
        "unit": "GCUPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "s16x2 (int16 lanes, exact)",
        "data": "synthetic",
        "config": {"workload": f"config {cfg.c} ({cfg.name}): {n_reads} reads x {m} bp per GPU vs {cfg.genome_len} bp genome, "
                               f"F={cfg.frag_len}, overlap={'m-1' if cfg.overlap < 0 else cfg.overlap}, both strands, top-2 + NW"
                               + ("" if args.mode == "plain" else f" [diagnostic mode: {args.mode}]")
                               + ("" if not n_with_n else f" [diagnostic: {n_with_n} reads carry one N]"),
                   "reads_per_gpu": n_reads, "read_len": m, "genome_bp": cfg.genome_len, "frag_len": cfg.frag_len,
                   "n_frag": G.n_frag, "reads_with_n": n_with_n,
                   "l2": f"flushed between steps (256 MiB write); packed genome + N mask = {genome_bytes / 1e6:.1f} MB "
                         + ("(L2-resident by design within a step)" if l2_resident else "(streams from HBM)"),
                   "parallelism": f"reads sharded over {world} GPU(s), genome replicated, no collective",
                   "launch": launch_info},
        "reads_per_s": n_reads * world / (ms_per_step * 1e-3),
        "scan_gcups": cells_step / (scan_avg_ms * 1e-3) / 1e9, "scan_ms": scan_avg_ms, "nw_ms": sum(nw_ms) / len(nw_ms),
        "genome_load_ms": genome_load_ms,
        "e2e": e2e,
        "gpu_launches": args.steps * (launch_info["launches"] + (0 if args.no_nw else 1) + (1 if args.mode == "pssm" else 0)),
        "clocks": clocks, "roofline": roofline,
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(cfg, genome, reads, lens)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def plumbing_only(args, cfg, rank: int, world: int) -> None:
    """The N > 1 host path of main() without a GPU: gloo process group, per-rank inputs, barrier, K "steps" whose device
    time is a rank-dependent sleep, max over ranks, rank 0 prints one JSON line.  Used by tests/test_bench_launch.py."""
    import hashlib
    import torch
    import torch.distributed as dist
    from paper_1403_2136_b200.shard import max_over_ranks
    if world > 1:
        dist.init_process_group("gloo")
    genome = gen.make_genome(20_000, cfg.genome_seed)[0]
    args.reads = args.reads or 64
    reads, lens, m, _ = rank_inputs(cfg, args, rank, world, genome)
    digest = hashlib.sha256(reads.tobytes()).hexdigest()[:16]
    if world > 1:
        dist.barrier()
    own_ms = 0.0
    for _ in range(args.steps):
        t0 = time.perf_counter()
        time.sleep(0.05 * (rank + 1))
        own_ms += 1e3 * (time.perf_counter() - t0)
    if world > 1:
        dist.barrier()
    total_ms = max_over_ranks(own_ms)
    digests = [digest]
    if world > 1:
        digests = [None] * world
        dist.all_gather_object(digests, digest)
    if rank == 0:
        print(json.dumps({"plumbing_only": True, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": total_ms / args.steps, "own_ms_rank0": own_ms, "reads_per_gpu": int(reads.shape[0]),
                          "read_digests": digests, "scaling": "weak"}), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
