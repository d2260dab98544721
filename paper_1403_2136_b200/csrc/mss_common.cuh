// Shared declarations of the CUDA side (product code; shares nothing with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/mss.h"

// Derived genome layout built by mss_genome_load (lives in the caller's workspace):
//   packed : 2-bit bases, padded with code 0 up to padded_bases
//   nmask  : 1 bit per base, 1 = N; every position >= n_bases is set, so kernels never bounds-check
// padded_bases = round_up(nfrag*F + MSS_MAX_READ_LEN + 128, 128): any window start in any fragment may read
// max_len bases forward without leaving the arrays.
struct mss_genome {
    const uint32_t* packed;      // device, in workspace
    const uint32_t* nmask;       // device, in workspace
    int64_t n_bases;
    int64_t padded_bases;
    int32_t frag_len;
    int32_t overlap;             // -1 = read length - 1
    int32_t n_frag;
    int device;
    int sm_count;
    int max_smem_optin;
};

struct ScanParams {
    const uint32_t* gpacked;
    const uint32_t* gnmask;
    int64_t n_bases;
    int32_t F, V, n_frag;
    const uint32_t* reads;
    const uint32_t* reads_nmask;   // nullable
    int32_t stride_words;
    const int32_t* lens;
    int32_t n_reads, max_len;
    int32_t match, mismatch;
    int32_t strands;               // MSS_FWD | MSS_REV
    int32_t zero;                  // always 0; a run-time zero the compiler cannot fold (DPX third operand)
    int32_t istep;                 // 1 = every read position; 2 = MaxSSmap_fast, every other position
    const uint32_t* pssm;          // nullable: per-read rows of (int16 pmatch | int16 pmismatch << 16) per position
    int32_t pssm_stride;           // words per row of pssm
    const uint16_t* ubound;        // nullable: pass-1 fragment score bounds [read][strand][fragment] (two-pass scan, pass 2)
    int32_t delta;                 // bound slack: a fragment's exact score lies in [ubound, ubound + delta]
};

// candidate of one fragment for one read: higher key = better under (score desc, strand asc, diag asc)
__host__ __device__ inline uint64_t frag_key(int32_t score, int32_t strand, int32_t diag)
{
    return ((uint64_t)(uint32_t)score << 32) | ((uint64_t)(1 - strand) << 31) | (uint64_t)(0x7FFFFFFF - diag);
}
__host__ __device__ inline void frag_key_unpack(uint64_t k, int32_t& score, int32_t& strand, int32_t& diag)
{
    score = (int32_t)(k >> 32);
    strand = 1 - (int32_t)((k >> 31) & 1);
    diag = 0x7FFFFFFF - (int32_t)(k & 0x7FFFFFFF);
}

// strictly-greater top-2 update while fragments arrive in ascending order (ties keep the lower fragment)
__device__ inline void top2_push(mss_hit_t& best, mss_hit_t& second, const mss_hit_t& h)
{
    if (best.frag < 0 || h.score > best.score) { second = best; best = h; }
    else if (second.frag < 0 || h.score > second.score) { second = h; }
}
// order-free merge of two candidates lists: a candidate beats another if (score desc, frag asc)
__device__ inline bool hit_better(const mss_hit_t& a, const mss_hit_t& b)
{
    if (a.frag < 0) return false;
    if (b.frag < 0) return true;
    if (a.score != b.score) return a.score > b.score;
    return a.frag < b.frag;
}
__device__ inline void top2_merge(mss_hit_t& best, mss_hit_t& second, const mss_hit_t& h)
{
    if (h.frag < 0) return;
    if (hit_better(h, best)) { second = best; best = h; }
    else if (hit_better(h, second)) { second = h; }
}

// base code 0..3, or 4 when masked as N
__device__ __forceinline__ uint32_t base_at(const uint32_t* packed, const uint32_t* nmask, int64_t p)
{
    uint32_t c = (packed[p >> 4] >> (2 * (uint32_t)(p & 15))) & 3u;
    uint32_t n = (nmask[p >> 5] >> (uint32_t)(p & 31)) & 1u;
    return n ? 4u : c;
}
// base of read r at position i of the strand-oriented query (strand 1 = reverse complement); 4 = N
__device__ __forceinline__ uint32_t read_base(const uint32_t* rw, const uint32_t* rn, int32_t m, int32_t i, int32_t strand)
{
    int32_t j = strand ? (m - 1 - i) : i;
    uint32_t c = (rw[j >> 4] >> (2 * (uint32_t)(j & 15))) & 3u;
    if (rn && ((rn[j >> 5] >> (uint32_t)(j & 31)) & 1u)) return 4u;
    return strand ? (3u - c) : c;
}

// records e for mss_last_cuda_error on this thread and returns MSS_ERR_CUDA (mss_api.cu)
int mss_record_cuda_error(cudaError_t e);

// launchers (each returns a cudaError_t)
cudaError_t launch_genome_prepare(const uint32_t* d_packed, const uint32_t* d_nmask, int64_t n_bases,
                                  int64_t padded_bases, uint32_t* out_packed, uint32_t* out_nmask, cudaStream_t st);

size_t scan_generic_workspace(const mss_genome* g, int32_t n_reads);
cudaError_t launch_scan_generic(const mss_genome* g, const ScanParams& p, void* ws, size_t ws_bytes,
                                mss_top2_t* d_out, cudaStream_t st, mss_launch_info_t* info);

size_t scan_dpx_workspace(const mss_genome* g, int32_t n_reads, int32_t max_len, int32_t strands);
bool scan_dpx_supported(const mss_genome* g, const ScanParams& p);
// per-position (pmatch, pmismatch) of the strand-oriented query: position i of the reverse-complemented read carries the
// scores of original position m-1-i (the quality belongs to the base call)
__device__ __forceinline__ uint32_t pssm_at(const uint32_t* row, int32_t m, int32_t i, int32_t strand)
{
    return row[strand ? (m - 1 - i) : i];
}
cudaError_t launch_scan_dpx(const mss_genome* g, const ScanParams& p, void* ws, size_t ws_bytes,
                            mss_top2_t* d_out, cudaStream_t st, mss_launch_info_t* info, int variant);

// two-pass scan (scan_filter.cu): bounded-error pass 1, then the exact kernel on the candidate fragments only
bool scan_filter_supported(const mss_genome* g, const ScanParams& p);
int32_t scan_filter_delta(const ScanParams& p);
void scan_filter_force_variant(int v, bool tile_kernel);
cudaError_t launch_scan_filter(const mss_genome* g, const ScanParams& p, uint16_t* ubound, cudaStream_t st, int32_t* grid_out,
                               int32_t* smem_out, int32_t* tile_out, int32_t* rpb_out, int32_t* kind_out);
// pass 1 in the lane-per-query layout (scan_filter_lq.cu): reads of up to 256 scored positions
bool scan_filter_lq_supported(const mss_genome* g, const ScanParams& p);
void scan_filter_lq_tune(int qsets, int half, int mode);
cudaError_t launch_scan_filter_lq(const mss_genome* g, const ScanParams& p, uint16_t* ubound, cudaStream_t st, int32_t* grid_out,
                                  int32_t* smem_out, int32_t* tile_out, int32_t* rpb_out, int32_t* kind_out);
size_t scan_two_pass_workspace(const mss_genome* g, int32_t n_reads, int32_t strands);
cudaError_t launch_scan_two_pass(const mss_genome* g, const ScanParams& p, void* ws, size_t ws_bytes,
                                 mss_top2_t* d_out, cudaStream_t st, mss_launch_info_t* info);

void scan_set_pass_timing(bool on);
void scan_set_two_pass_chunk_bytes(int64_t bytes);
cudaError_t scan_get_pass_times(float* pass1_ms, float* pass2_ms);

size_t nw_workspace(const mss_genome* g, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t pad);
cudaError_t launch_nw(const mss_genome* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t stride_words,
                      const int32_t* d_lens, int32_t n_reads, int32_t max_len, const mss_top2_t* d_hits,
                      const uint32_t* d_pssm, int32_t pssm_stride,
                      mss_scoring_t sc, int32_t pad, void* ws, size_t ws_bytes, cudaStream_t st,
                      int32_t* d_score, int64_t* d_ref_pos, uint32_t* d_cigar, int32_t cigar_stride, int32_t* d_n_cigar);

struct PssmLut { uint32_t v[94]; };   // phred 0..93 -> packed (pmatch, pmismatch), computed on the host in double
cudaError_t launch_pssm_build(const uint8_t* d_qual, int32_t qual_stride, const int32_t* d_lens, int32_t n_reads,
                              const PssmLut& lut, cudaStream_t st, uint32_t* d_pssm, int32_t pssm_stride);
cudaError_t launch_mapq(const mss_top2_t* d_hits, int32_t n_reads, double thr, cudaStream_t st, uint8_t* d_mapped, float* d_mapq);
cudaError_t run_dpx_probe(int32_t iters, cudaStream_t st, int sm_count, double* instr_per_s, float* ms);
cudaError_t run_pipe_probe(int which, int32_t iters, cudaStream_t st, int sm_count, double* per_clk_sm);
