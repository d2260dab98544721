"""paper_1403_2136_b200 -- B200-native MaxSSmap hot path (arXiv 1403.2136).

Thin Python binding of the C ABI in include/mss.h (libmss.so, hand-written CUDA for sm_100a).  The binding only
marshals arguments: every step of the path runs in the CUDA kernels.  PyTorch supplies device memory and streams.
There is no CPU fallback: importing works anywhere, but every compute call raises if libmss.so or a CUDA device is
missing.
"""
from .binding import (  # noqa: F401
    MSS_FWD, MSS_REV, MSS_BOTH, MSS_OVERLAP_PAPER, MssError, Scoring, Genome, lib, lib_path,
    mss_genome_load, mss_map_reads, mss_map_reads_fast, mss_map_reads_bounds, mss_map_reads_bounds_pssm, mss_pssm_build, mss_map_reads_pssm, mss_nw_align_pssm, pssm_bound,
    mss_map_reads_host, mss_map_align_host, mss_map_reads_static, mss_static_init, mss_static_scratch_bytes, MSS_ERR_STATIC_LIMIT, mss_nw_align, mss_mapq_filter,
    mss_set_scan_variant, mss_set_pass_timing, mss_set_pass1_geometry, mss_set_two_pass_chunk_bytes, mss_get_pass_times, mss_get_last_launch, mss_probe_dpx_peak, mss_probe_pipe, PROBE_NAMES, mss_strerror, declared_symbols,
)
