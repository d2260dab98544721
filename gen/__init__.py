"""Seeded synthetic inputs (genomes, reads) and the packed wire formats.

This module serves both the CPU oracle (oracle/) and the CUDA path
(paper_1403_2136_b200/): it holds *no* arithmetic of the method itself (no scoring,
no Kadane, no top-2, no alignment) -- only random draws, the read-simulation recipe
stated in DESIGN.md section 4 and the 2-bit / N-mask wire format of include/mss.h.
"""
from .synth import (  # noqa: F401
    A, C, G, T, N, S0,
    Config, CONFIGS, config,
    make_genome, make_reads, make_quals, revcomp,
    pack_2bit, unpack_2bit, pack_reads, sha256_of,
    decode, encode,
)
