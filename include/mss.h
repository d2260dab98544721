/*
 * mss.h -- C ABI of the B200-native MaxSSmap hot path (arXiv 1403.2136, Turki & Roshan).
 *
 * What the library computes (citations are /root/reference/PAPER.md lines; readings in DESIGN.md section 3):
 *
 *   mss_genome_load   PAPER.md:55, :69 (sections 2.2.1, 2.2.2): "MaxSSmap divides the genome into fragments of a
 *                     fixed size given by the user"; "if the genome is not a multiple of the fragment length we pad
 *                     the last fragment with N's"; the genome is transferred "just once".
 *   mss_map_reads     PAPER.md:41, :57 (sections 2.1.1, 2.2.1): for every read, the maximum scoring subsequence of
 *                     the per-base match/mismatch scores of the read laid gap-free at every window start of every
 *                     fragment ("sliding window", reading into neighbouring fragments to map across junctions);
 *                     "it outputs the fragment number with the highest and second highest score".
 *   mss_nw_align      PAPER.md:59, :91: "we align the read sequence with Needleman-Wunsch to the genome region from
 *                     the first part", match 5, mismatch -4, gap -26.
 *   mss_mapq_filter   PAPER.md:57, :63: mapped iff second/best < 0.9; MAPQ = -100 log2(second/best).
 *   mss_map_reads_fast   PAPER.md:93: MaxSSmap_fast, every other read nucleotide.
 *   mss_pssm_build, mss_map_reads_pssm, mss_nw_align_pssm   PAPER.md:61: base-quality position-specific scoring.
 *
 * Conventions
 *   - Every pointer named d_* is DEVICE memory owned by the caller; h_* is HOST memory owned by the caller.
 *     The library allocates no device memory: scratch comes from the caller through the *_workspace_bytes queries
 *     (mss_map_reads_static instead uses a static device array of MSS_STATIC_SCRATCH_BYTES that is part of the library image).
 *     mss_genome_load allocates one small host struct (the handle), released by mss_genome_free; the packed genome
 *     and the genome workspace must outlive the handle.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls enqueue work on it and
 *     return; outputs are valid once the caller has synchronised the stream.  The *_host entry points are the
 *     exception: they copy host buffers in, run, copy results out and synchronise before returning.
 *   - Return value: 0 (MSS_OK) or a negative mss_status.  No exception or abort crosses this boundary and there is
 *     no CPU fallback: without a CUDA device every compute call returns MSS_ERR_CUDA.
 *
 * Packed sequence format (genome and reads)
 *   base codes A=0 C=1 G=2 T=3 (complement = code XOR 3); base i sits in bits [2*(i%16), 2*(i%16)+2) of uint32 word
 *   i/16.  N mask: bit (i%32) of uint32 word i/32, 1 = N; the 2-bit code under an N is ignored.  A NULL mask means
 *   "no N".  Genome arrays hold ceil(n_bases/16) and ceil(n_bases/32) words.  Reads are rows of
 *   `read_stride_words` words (>= ceil(max_len/16)); their mask rows have ceil(read_stride_words/2) words; bits
 *   beyond len[r] are ignored.
 */
#ifndef MSS_H
#define MSS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mss_genome mss_genome_t;                          /* opaque handle */

typedef struct { int32_t match, mismatch, gap; } mss_scoring_t;  /* paper defaults 5, -4, -26;
                                                                    N against anything (N included) = mismatch */

typedef struct { int32_t frag, diag, score, strand; } mss_hit_t; /* frag: fragment index, -1 = no such fragment;
                                                                    diag: window start inside the fragment, [0, F);
                                                                    strand: 0 forward, 1 reverse-complemented read */
typedef struct { mss_hit_t best, second; } mss_top2_t;           /* 32 bytes per read */

enum { MSS_FWD = 1, MSS_REV = 2, MSS_BOTH = 3 };                 /* `strands` argument */
enum { MSS_OVERLAP_PAPER = -1 };                                 /* look-ahead = read length - 1, per read */

typedef enum {
    MSS_OK = 0,
    MSS_ERR_ARG = -1,        /* NULL pointer, n_bases <= 0, frag_len <= 0, overlap < -1, n_reads < 0, stride too small,
                                strands not in {1,2,3}, pad < 0, cigar_stride < 1 */
    MSS_ERR_RANGE = -2,      /* match <= 0, mismatch >= 0, gap >= 0, max_len*match > 32767, mismatch < -32768,
                                frag_len > 2^24, number of fragments > 2^31-1, max_len > MSS_MAX_READ_LEN */
    MSS_ERR_WORKSPACE = -3,  /* workspace_bytes smaller than the matching *_workspace_bytes query */
    MSS_ERR_CUDA = -4,       /* no device, launch failure, or any CUDA runtime error (see mss_last_cuda_error) */
    MSS_ERR_STATIC_LIMIT = -5 /* mss_map_reads_static: the batch needs more scratch than MSS_STATIC_SCRATCH_BYTES */
} mss_status;

#define MSS_MAX_READ_LEN 6553   /* floor(32767 / 5): packed 16-bit score lanes stay exact; checked against match */

/* ---- genome -------------------------------------------------------------------------------------------------- */

/* Bytes of device scratch mss_genome_load needs for a genome of n_bases (0 on bad arguments). */
size_t mss_genome_workspace_bytes(int64_t n_bases, int32_t frag_len, int32_t overlap);

/*
 * Derive the scan layout from the caller's packed genome.
 *   d_packed, d_nmask  packed genome and N mask (d_nmask may be NULL), n_bases bases.
 *   frag_len F >= 1    fragment f owns window starts [f*F, f*F+F); nfrag = ceil(n_bases/F); positions >= n_bases
 *                      behave as N.
 *   overlap V          bases past the fragment end a window may read: MSS_OVERLAP_PAPER (-1) = read length - 1
 *                      (the read is always "fully mapped"), V >= 0 = min(V, read length - 1).
 *   d_workspace        >= mss_genome_workspace_bytes(...) bytes, 16-byte aligned; owned by the caller, must outlive
 *                      the handle.
 * On success *out receives the handle.
 */
int mss_genome_load(const uint32_t *d_packed, const uint32_t *d_nmask, int64_t n_bases,
                    int32_t frag_len, int32_t overlap, void *d_workspace, size_t workspace_bytes,
                    void *stream, mss_genome_t **out);
int mss_genome_free(mss_genome_t *g);
int32_t mss_genome_num_fragments(const mss_genome_t *g);
int64_t mss_genome_num_bases(const mss_genome_t *g);

/* ---- first phase: MaxSS scan + top-2 -------------------------------------------------------------------------- */

size_t mss_map_workspace_bytes(const mss_genome_t *g, int32_t n_reads, int32_t max_len, int32_t strands);

/*
 * For every read r in [0, n_reads): score(f, strand, d) = max(0, best gap-free run) computed as
 *     H = 0; for i in [0, len[r]): stop if f*F+d+i >= f*F+F+Veff; H = max(0, H + s(read[i], genome[f*F+d+i])); best = max(best, H)
 * for every fragment f, enabled strand and window start d in [0,F); each fragment is represented by
 * its maximum (ties: forward strand first, then lowest d); d_out[r] = the two best *distinct* fragments (ties:
 * lowest fragment index; a fragment scoring 0 is still a fragment; with one fragment second.frag = -1).
 *   d_reads / d_reads_nmask / read_stride_words / d_lens: packed reads as described above, 1 <= len[r] <= max_len.
 *   max_len            upper bound of d_lens[] known to the host (sizes shared memory and the score-range check).
 *   sc                 match > 0 > mismatch; sc.gap is ignored here.
 *   strands            MSS_FWD, MSS_REV (reverse-complemented read against the forward genome) or MSS_BOTH.
 * Reads whose length lies outside [1, max_len] get best.frag = second.frag = -1.
 */
int mss_map_reads(const mss_genome_t *g, const uint32_t *d_reads, const uint32_t *d_reads_nmask,
                  int32_t read_stride_words, const int32_t *d_lens, int32_t n_reads, int32_t max_len,
                  mss_scoring_t sc, int32_t strands, void *d_workspace, size_t workspace_bytes,
                  void *stream, mss_top2_t *d_out);

/* ---- second phase: Needleman-Wunsch of each read against its best region --------------------------------------- */

size_t mss_nw_workspace_bytes(const mss_genome_t *g, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t pad);

/*
 * Fitting alignment (all of the read, any substring of the window; linear gap) of read r, reverse-complemented if
 * d_hits[r].best.strand = 1, against genome[ws, we): ws = max(0, f*F - pad), we = min(n_bases, f*F + F + Veff + pad),
 * f = d_hits[r].best.frag ("the region of the genome starting from the identified fragment and
 * spanning fragments to the right").  D[0][j] = 0, D[i][0] = i*gap,
 * D[i][j] = max(D[i-1][j-1] + s, D[i-1][j] + gap, D[i][j-1] + gap); score = max_j D[len][j], smallest such j;
 * traceback prefers diagonal (M, op 0), then up (I, op 1), then left (D, op 2).
 *   d_score[r], d_ref_pos[r] (0-based forward-genome position of the first window base used; ws + end column if
 *   none), d_cigar[r*cigar_stride ...] = BAM-style (len << 4 | op) in read order, d_n_cigar[r] = number of ops
 *   (ops beyond cigar_stride are counted but not written).  Reads with best.frag < 0: score 0, pos -1, 0 ops.
 */
int mss_nw_align(const mss_genome_t *g, const uint32_t *d_reads, const uint32_t *d_reads_nmask,
                 int32_t read_stride_words, const int32_t *d_lens, int32_t n_reads, int32_t max_len,
                 const mss_top2_t *d_hits, mss_scoring_t sc, int32_t pad,
                 void *d_workspace, size_t workspace_bytes, void *stream,
                 int32_t *d_score, int64_t *d_ref_pos, uint32_t *d_cigar, int32_t cigar_stride, int32_t *d_n_cigar);

/* ---- repeat filter and mapping quality ------------------------------------------------ */

/*
 * Per record ("considers the read to be mapped if the ratio of the second best to best score is below .9";
 * PAPER.md:63 MAPQ = -100 log2 p, p = second/best; PAPER.md:184 a stricter cutoff of 62):
 *   - best.frag < 0 or best.score <= 0: the ratio is undefined -> d_mapped[r] = 0, d_mapq[r] = 0 (reading 17);
 *   - p = second.score / best.score, second.score counting as 0 when second.frag < 0 (a genome of one fragment);
 *     p = 0 -> MAPQ = +infinity, else MAPQ = -100 log2 p, computed in IEEE double and stored as float32;
 *   - mapq_threshold < 0 (the default of the binding): the paper's rule in its exact form, mapped iff
 *     10*second < 9*best on the integers (the printed 15.2 is a rounded -100 log2 .9 = 15.2003 and would admit a ratio of
 *     exactly .9); mapq_threshold >= 0: mapped iff MAPQ > mapq_threshold, decided in double before the float32 store.
 * d_mapq may be NULL.
 */
int mss_mapq_filter(const mss_top2_t *d_hits, int32_t n_reads, double mapq_threshold,
                    void *stream, uint8_t *d_mapped, float *d_mapq);

/* ---- next rows: MaxSSmap_fast and base-quality position-specific scoring ------------------------------------------- */

/*
 * MaxSSmap_fast (section 2.3): "we consider every other nucleotides in the read sequence when mapping to
 * the genome".  Same arguments, output and errors as mss_map_reads; of the strand-oriented read only positions
 * i = 0, 2, 4, ... are scored (each still against genome[f*F+d+i]) and the maximum scoring subsequence is taken over
 * that sub-sequence of scores (reading 20).  Workspace: mss_map_workspace_bytes.
 */
int mss_map_reads_fast(const mss_genome_t *g, const uint32_t *d_reads, const uint32_t *d_reads_nmask,
                       int32_t read_stride_words, const int32_t *d_lens, int32_t n_reads, int32_t max_len,
                       mss_scoring_t sc, int32_t strands, void *d_workspace, size_t workspace_bytes,
                       void *stream, mss_top2_t *d_out);

/*
 * Position-specific scoring matrix from base qualities (section 2.2.1): "let x be the probability that
 * the base at position i is correctly sequenced ... The score of a match against the nucleotide at position i is
 * match x x and mismatch is mismatch x x/3."  x = 1 - 10^(-Q/10) for phred quality Q.  The paper keeps floats; here
 * the table is fixed point with `scale` units per score point (reading 22):
 *     pmatch = round(scale*match*x), pmismatch = round(scale*mismatch*x/3)   (IEEE double, halves away from zero)
 *   d_qual             phred values (0..93; larger values count as 93), rows of qual_stride bytes, read order
 *   d_pssm             out: rows of pssm_stride uint32 per read, entry i = (uint16)pmatch_i | (uint16)pmismatch_i << 16
 *                      (two int16); entries at or beyond len[r] are 0
 *   scale >= 1         scale*match <= 32767, scale*mismatch >= -32768, else MSS_ERR_RANGE
 * A caller may also fill d_pssm itself with any table satisfying pmismatch_i <= 0 <= pmatch_i.
 */
int mss_pssm_build(const uint8_t *d_qual, int32_t qual_stride, const int32_t *d_lens, int32_t n_reads,
                   mss_scoring_t sc, int32_t scale, void *stream, uint32_t *d_pssm, int32_t pssm_stride);

/*
 * mss_map_reads with s(read[i], genome base) replaced by the read's own table: pmatch_i if the bases are equal (and
 * neither is N) else pmismatch_i; on the reverse strand position i of the reverse-complemented read carries the
 * entry of original position len-1-i.  `bound` states the table's range for the 16-bit lane check and for the slack
 * of the two-pass scan's bounds (min(PM, -PMM) - PMM: a tight bound prunes better): bound.match >= every pmatch_i,
 * bound.mismatch <= every pmismatch_i (for a table from mss_pssm_build: {scale*match, -ceil(scale*|mismatch|/3),
 * scale*gap}); max_len*bound.match <= 32767 else MSS_ERR_RANGE; entries outside the stated bound give undefined
 * scores.  pssm_stride >= max_len.  Workspace: mss_map_workspace_bytes.  The scan is the two-pass scan where the geometry
 * allows it (pass 1: scan_filter_lq_kernel in its PSSM form), else the exact kernel on every fragment.
 */
int mss_map_reads_pssm(const mss_genome_t *g, const uint32_t *d_reads, const uint32_t *d_reads_nmask,
                       int32_t read_stride_words, const int32_t *d_lens, int32_t n_reads, int32_t max_len,
                       const uint32_t *d_pssm, int32_t pssm_stride, mss_scoring_t bound, int32_t strands,
                       void *d_workspace, size_t workspace_bytes, void *stream, mss_top2_t *d_out);

/*
 * mss_nw_align with the same per-position scores ("in both phases of the program"); bound.gap is the
 * gap cost in the table's units (scale*gap).  Workspace: mss_nw_workspace_bytes(g, n_reads, max_len, bound, pad).
 */
int mss_nw_align_pssm(const mss_genome_t *g, const uint32_t *d_reads, const uint32_t *d_reads_nmask,
                      int32_t read_stride_words, const int32_t *d_lens, int32_t n_reads, int32_t max_len,
                      const mss_top2_t *d_hits, const uint32_t *d_pssm, int32_t pssm_stride, mss_scoring_t bound,
                      int32_t pad, void *d_workspace, size_t workspace_bytes, void *stream,
                      int32_t *d_score, int64_t *d_ref_pos, uint32_t *d_cigar, int32_t cigar_stride, int32_t *d_n_cigar);

/* ---- end-to-end convenience with HOST buffers (used for the e2e timing of bench.py) ---------------------------- */

/*
 * Same as mss_map_reads, but reads, lengths and output are HOST pointers: copies them to the device workspace,
 * scans, copies the n_reads records back and synchronises.  d_workspace must hold
 * mss_map_host_workspace_bytes(...) bytes.
 */
size_t mss_map_host_workspace_bytes(const mss_genome_t *g, int32_t n_reads, int32_t max_len, int32_t read_stride_words,
                                    int32_t strands);
int mss_map_reads_host(const mss_genome_t *g, const uint32_t *h_reads, const uint32_t *h_reads_nmask,
                       int32_t read_stride_words, const int32_t *h_lens, int32_t n_reads, int32_t max_len,
                       mss_scoring_t sc, int32_t strands, void *d_workspace, size_t workspace_bytes,
                       void *stream, mss_top2_t *h_out);

/*
 * Both phases with HOST buffers: reads in; top-2 records, NW score, position and CIGAR out (all h_* pointers are
 * host memory, pinned for full copy speed).  Copies in, mss_map_reads, mss_nw_align on the best hits, copies out,
 * synchronises.  d_workspace must hold mss_map_align_host_workspace_bytes(...) bytes.
 */
size_t mss_map_align_host_workspace_bytes(const mss_genome_t *g, int32_t n_reads, int32_t max_len,
                                          int32_t read_stride_words, int32_t strands, mss_scoring_t sc, int32_t pad,
                                          int32_t cigar_stride);
int mss_map_align_host(const mss_genome_t *g, const uint32_t *h_reads, const uint32_t *h_reads_nmask,
                       int32_t read_stride_words, const int32_t *h_lens, int32_t n_reads, int32_t max_len,
                       mss_scoring_t sc, int32_t strands, int32_t pad, void *d_workspace, size_t workspace_bytes,
                       void *stream, mss_top2_t *h_top2, int32_t *h_score, int64_t *h_ref_pos, uint32_t *h_cigar,
                       int32_t cigar_stride, int32_t *h_n_cigar);

/* ---- diagnostics ------------------------------------------------------------------------------------------------ */

const char *mss_strerror(int status);
int mss_last_cuda_error(void);                 /* cudaError_t of the last MSS_ERR_CUDA on this thread, 0 if none */
int mss_version(void);                         /* 100*major + minor */

/*
 * mss_map_reads without a caller workspace, for callers that cannot allocate or hand over device scratch (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same inputs, same records, same kernels as
 * mss_map_reads; the scan's scratch lives in a static device array of MSS_STATIC_SCRATCH_BYTES inside the
 * library, which every GPU that loads the library holds until the process exits.  The call allocates nothing (no cudaMalloc,
 * cudaFree or allocating library routine) and only enqueues work on `stream`.
 *   limit      mss_map_workspace_bytes(g, n_reads, max_len, strands) <= MSS_STATIC_SCRATCH_BYTES, else MSS_ERR_STATIC_LIMIT
 *              (nothing is launched): at the E. coli-sized geometry (1124 fragments, both strands) about 3,700 reads per call
 *              (the query is the maximum over every scan path: 8 B per read and fragment for the generic kernel);
 *              larger batches go through mss_map_reads, or in several calls.
 *   sharing    every call on a device uses the SAME array, which keeps the previous call's contents.  Nothing in it has to start
 *              at zero (every bound / partial record is written before it is read), so no clearing is needed -- but two calls
 *              whose kernels overlap on the GPU (different streams, or concurrent graphs) race on it: serialise them.
 *   set-up     mss_static_init(), once per device with that device current, resolves the array's device address
 *              (cudaGetSymbolAddress; this is also where a lazily loaded module is brought in).  mss_map_reads_static does it
 *              on first use if it was not called; callers that capture graphs call it before capture.
 * Other errors as mss_map_reads.  mss_static_scratch_bytes() returns MSS_STATIC_SCRATCH_BYTES.
 */
#define MSS_STATIC_SCRATCH_BYTES (32u << 20)
size_t mss_static_scratch_bytes(void);
int mss_static_init(void);
int mss_map_reads_static(const mss_genome_t *g, const uint32_t *d_reads, const uint32_t *d_reads_nmask,
                         int32_t read_stride_words, const int32_t *d_lens, int32_t n_reads, int32_t max_len,
                         mss_scoring_t sc, int32_t strands, void *stream, mss_top2_t *d_out);

/*
 * Tuning / introspection (does not change results): select the scan kernel variant (0 = automatic: the two-pass scan
 * where the geometry allows it, else the one-pass tile kernel, else the generic kernel; 1 = generic; 2-6 = one-pass tile
 * kernels (K, T) = (8,256), (8,128), (8,64), (4,256), (16,128); 7 = two-pass, same as automatic: pass 1 is the
 * lane-per-query kernel for reads of up to 256 scored positions, else the tile kernel; 8-12 = two-pass with pass 1 = the
 * tile kernel and its tile (K, T) = (4,256), (4,128), (4,64), (8,128), (8,256) forced; 13 = two-pass with the tile kernel
 * and its own choice of tile; anything else: MSS_ERR_ARG) and report the
 * launch geometry of the last mss_map_reads call on this thread (two-pass: variant 7, grid / smem_bytes / tile_diagonals of
 * pass 1, block 0, launches = 2 per chunk of reads).  Used by bench.py and the parity tests to cover every variant.
 * Every tuning switch of this section (scan variant, forced pass-1 tile, pass timing, bounds chunk size, queries per
 * pass-1 block) is thread-local: it affects only calls made later on the same host thread.
 */
int mss_set_scan_variant(int variant);
typedef struct {
    int32_t variant, grid, block, smem_bytes, reads_per_block, tile_diagonals, launches;
    int32_t pass1_kernel;   /* two-pass scan: 1 = tile kernel, 2 / 3 / 4 = lane-per-query kernel with int16 DPX / fp16 / e5m2 operands and the
                               plane offsets in registers, 6 / 7 / 8 = the same with the offsets in a shared-memory table, 5 = its PSSM form; else 0 */
} mss_launch_info_t;
int mss_get_last_launch(mss_launch_info_t *out);

/*
 * Per-pass device times of the two-pass scan, for the roofline of bench.py: after mss_set_pass_timing(1) every
 * mss_map_reads / mss_map_reads_fast call on this thread that takes the two-pass path records CUDA events on its stream
 * before pass 1, between the passes and after pass 2 (per chunk of reads); mss_get_pass_times waits for the last event
 * of the latest such call and returns the summed milliseconds (0, 0 if that call took another path).
 */
int mss_set_pass_timing(int on);
/* Bytes of pass-1 bounds produced per chunk of reads (default 256 MiB, <= 0 restores it; this thread only).  The workspace
 * queries follow it.  Results do not depend on it; tests set it small to exercise the chunk loop. */
int mss_set_two_pass_chunk_bytes(int64_t bytes);
/* Geometry of the lane-per-query pass-1 kernel (this thread only; results do not depend on it).  query_sets: 32-query
 * sets per block, 1, 2 or 4 (reads per block = 16, 32 or 64 with both strands, twice that with one; 0 = automatic) --
 * BASELINE.json config 5's "reads-per-block swept".  tile_window_starts: window starts per tile (even; 0 = automatic:
 * the tile with the least padding of the fragment length that leaves room for two blocks per SM); a value no tile can
 * take makes pass 1 fall back to the tile kernel.  arithmetic: how the chains are computed -- 0 = packed int16 DPX
 * (VIADDMNMX.S16x2.RELU), 1 = fp16 pairs (HFMA2.RELU; exact, every value is an integer <= 2048), 2 = e5m2 operand bytes
 * widened to fp16 pairs (half the shared-memory traffic), -1 = automatic: the highest of these the scoring and the read
 * length allow (a forced value that they do not allow is lowered the same way).  Adding 8 (8..10, 11 = automatic arithmetic)
 * makes the kernel read a query's plane offsets from its shared-memory table instead of registers, adding 16 (16..19) keeps
 * them in registers where the read length allows (up to 256 scored positions); default: registers up to 152 scored positions.
 * Adding 32 (32..35) keeps 8 chains per thread where the default is 16 (reads of up to 52 and of 65-76 scored positions, and the
 * table-driven instance).  query_sets 0 = the most sets with which read groups x fragments still fill the GPU.
 * Bad values: MSS_ERR_ARG. */
int mss_set_pass1_geometry(int32_t query_sets, int32_t tile_window_starts, int32_t arithmetic);
int mss_get_pass_times(float *h_pass1_ms, float *h_pass2_ms);

/*
 * Pass 1 of the two-pass scan on its own (scan variant 7): for every read, enabled strand and fragment
 * a 16-bit lower bound u of the fragment's exact MaxSS score with  u <= score <= u + *h_delta  (two Kadane steps per
 * DPX instruction, H sampled after every second step), or 0xFFFF = "not bounded" (reads holding an N, bad lengths).
 * d_bounds holds n_reads * (strands == MSS_BOTH ? 2 : 1) * n_fragments uint16, indexed [read][strand][fragment];
 * every_other != 0 bounds the MaxSSmap_fast scores instead.  MSS_ERR_RANGE if the geometry has no two-pass path
 * (fewer than 8 fragments, frag_len < 256, 2*match or 2*mismatch outside int16).  mss_map_reads itself uses these
 * bounds only to skip fragments that cannot reach a read's top-2; its records are those of the one-pass scan.
 * Reads holding an N are bounded like any other by the lane-per-query kernel; the tile kernel marks them 0xFFFF.
 * mss_map_reads_bounds_pssm: the same for base-quality scoring (table and `bound` as for mss_map_reads_pssm); *h_delta
 * = min(bound.match, -bound.mismatch) - bound.mismatch.
 */
int mss_map_reads_bounds(const mss_genome_t *g, const uint32_t *d_reads, const uint32_t *d_reads_nmask,
                         int32_t read_stride_words, const int32_t *d_lens, int32_t n_reads, int32_t max_len,
                         mss_scoring_t sc, int32_t strands, int32_t every_other, void *stream,
                         uint16_t *d_bounds, int32_t *h_delta);
int mss_map_reads_bounds_pssm(const mss_genome_t *g, const uint32_t *d_reads, const uint32_t *d_reads_nmask,
                              int32_t read_stride_words, const int32_t *d_lens, int32_t n_reads, int32_t max_len,
                              const uint32_t *d_pssm, int32_t pssm_stride, mss_scoring_t bound, int32_t strands,
                              void *stream, uint16_t *d_bounds, int32_t *h_delta);

/*
 * Live measurement of the integer/DPX issue peak the scan's roofline is quoted against: runs `iters` dependent
 * rounds of 8 independent VIADDMNMX.S16x2.RELU / VIMNMX3.S16x2 chains (2:1 mix, the scan's own DPX mix) per thread
 * on every SM and returns thread-instructions per second in *h_instr_per_s and the elapsed ms in *h_ms.
 */
int mss_probe_dpx_peak(int32_t iters, void *stream, double *h_instr_per_s, float *h_ms);

/*
 * Issue-rate probes behind the roofline denominators: `which` selects an instruction or mix, the result
 * is thread-instructions (row 4: cells) per clock per SM, measured with clock64 over `iters` rounds of 64 chain steps on
 * 1024 threads per SM.  0 VIADDMNMX.S16x2.RELU, 1 VIMNMX3.S16x2, 2 their 2:1 mix, 3 LDS.32 conflict-free (x 4 B = the
 * shared-memory feed), 4 the exact scan's inner mix (LDS.32 + VIADDMNMX per 2 cells + VIMNMX3 per 4 cells).
 * Synchronises the stream before returning.  (The design-experiment rows of round 1 are no longer part of the library.)
 */
enum { MSS_PROBE_COUNT = 5 };
int mss_probe_pipe(int32_t which, int32_t iters, void *stream, double *h_per_clk_sm);

#ifdef __cplusplus
}
#endif
#endif /* MSS_H */
