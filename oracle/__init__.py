"""CPU oracle -- TEST INFRASTRUCTURE ONLY (see oracle/maxss_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this
package.  The product (paper_1403_2136_b200) never does."""
from . import oracle  # noqa: F401
from .oracle import build, map_reads, fragment_scores, nw_align, map_reads_parallel, diagonal_score  # noqa: F401
from .oracle import pssm_from_phred, map_reads_pssm, map_reads_pssm_parallel, nw_align_pssm, mapq_filter  # noqa: F401
