// a7: Needleman-Wunsch second stage -- placeholder until the kernel lands.
#include "mss_common.cuh"

size_t nw_workspace(const mss_genome* g, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t pad) { return 256; }
cudaError_t launch_nw(const mss_genome* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t stride_words,
                      const int32_t* d_lens, int32_t n_reads, int32_t max_len, const mss_top2_t* d_hits,
                      mss_scoring_t sc, int32_t pad, void* ws, size_t ws_bytes, cudaStream_t st,
                      int32_t* d_score, int64_t* d_ref_pos, uint32_t* d_cigar, int32_t cigar_stride, int32_t* d_n_cigar)
{
    return cudaErrorNotSupported;
}
