/*
 * oracle/maxss_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded CPU statement of what MaxSSmap's hot path computes, written from the
 * paper's text (arXiv 1403.2136, /root/reference/PAPER.md) and the readings fixed in DESIGN.md section 3.
 * It shares no code with the CUDA path (paper_1403_2136_b200/csrc): no common headers, helpers or tables.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Everything is int32 arithmetic on unpacked base codes (0=A 1=C 2=G 3=T 4=N), loops in the paper's order:
 * fragment -> window start (diagonal) -> read position.  No blocking, no SIMD, no look-ahead.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute force over all gap-free substring pairs, closed
 * forms (exact read = m*match, truncated prefix), reverse-complement symmetry, whole-genome = max over
 * fragments for every F, tie-break constructions, Fig. 2 fragment cutting, exhaustive
 * enumeration of all fitting alignments for NW, planted-indel CIGARs.  The next-row functions at the end of the file
 * (MaxSSmap_fast, base-quality position-specific scoring) are pinned in tests/test_oracle_next_pins.py: brute force
 * over every scored sub-range, the decimated-sequence reduction to the pinned plain scan, the uniform-score reduction
 * to the pinned plain functions, closed-form phred values, exhaustive NW enumeration.  oracle_mapq_filter (repeat filter +
 * MAPQ) is pinned in tests/test_oracle_mapq_pins.py: the paper's printed pairs (.9 <-> 15.2, threshold 62), exact rational
 * comparison for the .9 rule, closed forms at ratios 2^-k, the inverse relation through exact integer powers, edge readings.
 * Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { int32_t frag, diag, score, strand; } ohit_t;   /* strand 0 = forward, 1 = reverse */

/* substitution score: "a substitution scoring matrix, or a trivial match or mismatch cost" (PAPER.md:41,
 * section 2.1.1); N against anything, N included, is a mismatch (reading 6; the paper's profile has
 * an N row).  Held as the 5x5 matrix over {A,C,G,T,N} the paper speaks of. */
typedef struct { int32_t s[5][5]; } submat_t;

static submat_t make_submat(int32_t match, int32_t mismatch)
{
    submat_t M;
    for (int a = 0; a < 5; a++)
        for (int b = 0; b < 5; b++)
            M.s[a][b] = (a < 4 && a == b) ? match : mismatch;
    return M;
}

/* Genome extended with N beyond its end: "If the genome is not a multiple of the fragment length we pad the
 * last fragment with N's" (section 2.2.2); `extra` more N so that a window may hang off the end. */
static uint8_t *padded_genome(const uint8_t *genome, int64_t G, int64_t padded_len)
{
    uint8_t *gp = (uint8_t *)malloc((size_t)padded_len);
    memcpy(gp, genome, (size_t)G);
    memset(gp + G, 4, (size_t)(padded_len - G));
    return gp;
}

/* Maximum scoring subsequence of the substitution scores of read r (length m) laid gap-free on the padded
 * genome with r[0] at position g, reading no genome position >= end ("the contiguous
 * subsequence that maximizes the sum"; the linear-time scan of [15]).  The empty subsequence scores 0. */
static int32_t maxss_diagonal(const uint8_t *gp, int64_t g, int64_t end,
                              const uint8_t *r, int32_t m, const submat_t *M)
{
    int32_t H = 0, best = 0;
    int32_t n = (end - g < m) ? (int32_t)(end - g) : m;    /* read positions whose genome base is readable */
    for (int32_t i = 0; i < n; i++) {
        H += M->s[r[i]][gp[g + i]];
        if (H < 0) H = 0;
        if (H > best) best = H;
    }
    return best;
}

static void reverse_complement(const uint8_t *r, int32_t m, uint8_t *out)
{
    for (int32_t i = 0; i < m; i++) {
        uint8_t c = r[m - 1 - i];
        out[i] = c < 4 ? (uint8_t)(3 - c) : 4;
    }
}

/*
 * First phase (section 2.2.1): the genome is cut into nfrag = ceil(G/F) disjoint fragments of
 * length F; the read slides over every window start d in [0,F) of fragment f (global start g = f*F+d, Fig. 1
 * PAPER.md:271 "slides it across fragment 0, and stops when it has covered all of fragment 0"), reading into
 * the neighbouring fragments up to V bases past the fragment end ("each thread also considers neighboring
 * fragments"); the fragment's score is the maximum over its window starts (and enabled strands); the output is
 * "the fragment number with the highest and second highest score".
 *   V = -1: look-ahead m-1 (read always fully laid out); V >= 0: min(V, m-1).
 *   strands: bit 0 = forward, bit 1 = reverse-complemented read against the forward genome.
 * Ties: first maximiser in the order strand (fwd, rev) then d ascending within a fragment; lowest fragment
 * index between fragments (strictly-greater replacement while f ascends).
 * out[2*r] = best, out[2*r+1] = second; "no such fragment" = {-1,0,0,0}.
 */
void oracle_map_reads(const uint8_t *genome, int64_t G, int32_t F, int32_t V,
                      const uint8_t *reads, int32_t read_stride, const int32_t *lens, int32_t n_reads,
                      int32_t match, int32_t mismatch, int32_t strands, ohit_t *out)
{
    int64_t nfrag = (G + F - 1) / F;
    int32_t max_m = 0;
    for (int32_t r = 0; r < n_reads; r++) if (lens[r] > max_m) max_m = lens[r];
    uint8_t *gp = padded_genome(genome, G, nfrag * F + max_m);
    submat_t M = make_submat(match, mismatch);
    for (int32_t r = 0; r < n_reads; r++) {
        int32_t m = lens[r];
        const uint8_t *fwd = reads + (int64_t)r * read_stride;
        uint8_t *rev = (uint8_t *)malloc((size_t)(m > 0 ? m : 1));
        reverse_complement(fwd, m, rev);
        int32_t Veff = (V < 0 || V > m - 1) ? m - 1 : V;
        ohit_t best = { -1, 0, 0, 0 }, second = { -1, 0, 0, 0 };
        for (int64_t f = 0; f < nfrag; f++) {
            int64_t end = f * F + F + Veff;
            ohit_t fb = { (int32_t)f, 0, -1, 0 };             /* score -1 = nothing seen yet */
            for (int32_t s = 0; s < 2; s++) {
                if (!(strands & (1 << s))) continue;
                const uint8_t *q = s ? rev : fwd;
                for (int32_t d = 0; d < F; d++) {
                    int32_t sc = maxss_diagonal(gp, f * F + d, end, q, m, &M);
                    if (sc > fb.score) { fb.score = sc; fb.diag = d; fb.strand = s; }
                }
            }
            if (best.frag < 0 || fb.score > best.score) { second = best; best = fb; }
            else if (second.frag < 0 || fb.score > second.score) { second = fb; }
        }
        out[2 * r] = best;
        out[2 * r + 1] = second;
        free(rev);
    }
    free(gp);
}

/* Per-fragment scores of one read on one strand (test helper for the invariants: every fragment's
 * (score, first-maximising d)). strand 0 uses r, 1 its reverse complement. */
void oracle_fragment_scores(const uint8_t *genome, int64_t G, int32_t F, int32_t V,
                            const uint8_t *r, int32_t m, int32_t match, int32_t mismatch, int32_t strand,
                            int32_t *score_out, int32_t *diag_out)
{
    int64_t nfrag = (G + F - 1) / F;
    uint8_t *gp = padded_genome(genome, G, nfrag * F + m);
    submat_t M = make_submat(match, mismatch);
    uint8_t *q = (uint8_t *)malloc((size_t)(m > 0 ? m : 1));
    if (strand) reverse_complement(r, m, q); else memcpy(q, r, (size_t)m);
    int32_t Veff = (V < 0 || V > m - 1) ? m - 1 : V;
    for (int64_t f = 0; f < nfrag; f++) {
        int32_t bs = -1, bd = 0;
        for (int32_t d = 0; d < F; d++) {
            int32_t sc = maxss_diagonal(gp, f * F + d, f * F + F + Veff, q, m, &M);
            if (sc > bs) { bs = sc; bd = d; }
        }
        score_out[f] = bs; diag_out[f] = bd;
    }
    free(q); free(gp);
}

/* One window start on its own (test helper): the score of global window start g = f*F+d under the same
 * look-ahead rule as oracle_map_reads. */
int32_t oracle_diagonal_score(const uint8_t *genome, int64_t G, int32_t F, int32_t V, int64_t g,
                              const uint8_t *r, int32_t m, int32_t match, int32_t mismatch)
{
    int64_t nfrag = (G + F - 1) / F;
    uint8_t *gp = padded_genome(genome, G, nfrag * F + m);
    submat_t M = make_submat(match, mismatch);
    int32_t Veff = (V < 0 || V > m - 1) ? m - 1 : V;
    int64_t f = g / F;
    int32_t sc = maxss_diagonal(gp, g, f * F + F + Veff, r, m, &M);
    free(gp);
    return sc;
}

/*
 * Second phase (section 2.2.1; scores PAPER.md:91): "we align the read sequence with
 * Needleman-Wunsch to the genome region from the first part", match 5, mismatch -4, gap -26 (linear).
 * Region (readings 14-16): window W = genome[ws, we), ws = max(0, f*F - pad),
 * we = min(G, f*F + F + Veff + pad) around the best fragment f; the alignment is *fitting*: all of the read
 * (reverse-complemented when the hit is on the reverse strand), any substring of W:
 *     D[0][j] = 0, D[i][0] = i*gap,
 *     D[i][j] = max(D[i-1][j-1] + s(Q[i-1], W[j-1]), D[i-1][j] + gap, D[i][j-1] + gap).
 * score = max_j D[m][j], end column = smallest such j.  Traceback from (m, j*) to row 0 taking at every cell
 * the first move that reproduces D[i][j] in the order diagonal ('M', op 0), up ('I', op 1, consumes a read
 * base), left ('D', op 2, consumes a genome base).  ref_pos = ws + (column at which row 0 is reached).
 * CIGAR: run-length, read order, BAM encoding len<<4|op.  A read with hit.frag < 0 gets score 0, pos -1, no ops.
 */
void oracle_nw_align(const uint8_t *genome, int64_t G, int32_t F, int32_t V,
                     const uint8_t *reads, int32_t read_stride, const int32_t *lens, int32_t n_reads,
                     const ohit_t *top2 /* 2 per read */, int32_t match, int32_t mismatch, int32_t gap, int32_t pad,
                     int32_t *score_out, int64_t *pos_out, uint32_t *cigar_out, int32_t cigar_stride, int32_t *ncig_out)
{
    submat_t M = make_submat(match, mismatch);
    for (int32_t r = 0; r < n_reads; r++) {
        ohit_t h = top2[2 * r];
        int32_t m = lens[r];
        if (h.frag < 0) { score_out[r] = 0; pos_out[r] = -1; ncig_out[r] = 0; continue; }
        uint8_t *q = (uint8_t *)malloc((size_t)m);
        if (h.strand) reverse_complement(reads + (int64_t)r * read_stride, m, q);
        else memcpy(q, reads + (int64_t)r * read_stride, (size_t)m);
        int32_t Veff = (V < 0 || V > m - 1) ? m - 1 : V;
        int64_t ws = (int64_t)h.frag * F - pad;           if (ws < 0) ws = 0;
        int64_t we = (int64_t)h.frag * F + F + Veff + pad; if (we > G) we = G;
        int64_t L = we - ws;
        int64_t cols = L + 1;
        int32_t *D = (int32_t *)malloc(sizeof(int32_t) * (size_t)(m + 1) * (size_t)cols);
        for (int64_t j = 0; j <= L; j++) D[j] = 0;
        for (int32_t i = 1; i <= m; i++) {
            D[(int64_t)i * cols] = i * gap;
            for (int64_t j = 1; j <= L; j++) {
                int32_t dg = D[(int64_t)(i - 1) * cols + j - 1] + M.s[q[i - 1]][genome[ws + j - 1]];
                int32_t up = D[(int64_t)(i - 1) * cols + j] + gap;
                int32_t lf = D[(int64_t)i * cols + j - 1] + gap;
                int32_t v = dg;
                if (up > v) v = up;
                if (lf > v) v = lf;
                D[(int64_t)i * cols + j] = v;
            }
        }
        int64_t jbest = 0;
        for (int64_t j = 1; j <= L; j++)
            if (D[(int64_t)m * cols + j] > D[(int64_t)m * cols + jbest]) jbest = j;
        score_out[r] = D[(int64_t)m * cols + jbest];
        /* traceback, ops collected end-to-start */
        uint8_t *ops = (uint8_t *)malloc((size_t)(m + L + 1));
        int64_t nops = 0;
        int32_t i = m; int64_t j = jbest;
        while (i > 0) {
            int32_t v = D[(int64_t)i * cols + j];
            if (j > 0 && D[(int64_t)(i - 1) * cols + j - 1] + M.s[q[i - 1]][genome[ws + j - 1]] == v) {
                ops[nops++] = 0; i--; j--;
            } else if (D[(int64_t)(i - 1) * cols + j] + gap == v) {
                ops[nops++] = 1; i--;
            } else {
                ops[nops++] = 2; j--;
            }
        }
        pos_out[r] = ws + j;
        int32_t nc = 0;
        uint32_t *cg = cigar_out + (int64_t)r * cigar_stride;
        for (int64_t k = nops - 1; k >= 0; ) {
            uint8_t op = ops[k]; uint32_t len = 0;
            while (k >= 0 && ops[k] == op) { len++; k--; }
            if (nc < cigar_stride) cg[nc] = (len << 4) | op;
            nc++;
        }
        ncig_out[r] = nc;
        free(ops); free(D); free(q);
    }
}

/* ====================================================================================================================
 * Next rows: MaxSSmap_fast and base-quality position-specific scoring.  Same rules as above: plain
 * loops in the paper's order, int32 arithmetic, nothing shared with the CUDA path.
 * ==================================================================================================================== */

/*
 * MaxSSmap_fast (section 2.3): "we consider every other nucleotides in the read sequence when mapping to
 * the genome".  Reading (reading 20): of the strand-oriented query as it is slid over the genome, only
 * positions i = 0, 2, 4, ... are scored, each against genome position g+i as before; the maximum scoring subsequence is
 * taken over that sub-sequence of scores.  Everything else (fragments, look-ahead, ties, top-2) is oracle_map_reads.
 */
static int32_t maxss_diagonal_every_other(const uint8_t *gp, int64_t g, int64_t end,
                                          const uint8_t *r, int32_t m, const submat_t *M)
{
    int32_t H = 0, best = 0;
    int32_t n = (end - g < m) ? (int32_t)(end - g) : m;
    for (int32_t i = 0; i < n; i += 2) {
        H += M->s[r[i]][gp[g + i]];
        if (H < 0) H = 0;
        if (H > best) best = H;
    }
    return best;
}

void oracle_map_reads_fast(const uint8_t *genome, int64_t G, int32_t F, int32_t V,
                           const uint8_t *reads, int32_t read_stride, const int32_t *lens, int32_t n_reads,
                           int32_t match, int32_t mismatch, int32_t strands, ohit_t *out)
{
    int64_t nfrag = (G + F - 1) / F;
    int32_t max_m = 0;
    for (int32_t r = 0; r < n_reads; r++) if (lens[r] > max_m) max_m = lens[r];
    uint8_t *gp = padded_genome(genome, G, nfrag * F + max_m);
    submat_t M = make_submat(match, mismatch);
    for (int32_t r = 0; r < n_reads; r++) {
        int32_t m = lens[r];
        const uint8_t *fwd = reads + (int64_t)r * read_stride;
        uint8_t *rev = (uint8_t *)malloc((size_t)(m > 0 ? m : 1));
        reverse_complement(fwd, m, rev);
        int32_t Veff = (V < 0 || V > m - 1) ? m - 1 : V;
        ohit_t best = { -1, 0, 0, 0 }, second = { -1, 0, 0, 0 };
        for (int64_t f = 0; f < nfrag; f++) {
            int64_t end = f * F + F + Veff;
            ohit_t fb = { (int32_t)f, 0, -1, 0 };
            for (int32_t s = 0; s < 2; s++) {
                if (!(strands & (1 << s))) continue;
                const uint8_t *q = s ? rev : fwd;
                for (int32_t d = 0; d < F; d++) {
                    int32_t sc = maxss_diagonal_every_other(gp, f * F + d, end, q, m, &M);
                    if (sc > fb.score) { fb.score = sc; fb.diag = d; fb.strand = s; }
                }
            }
            if (best.frag < 0 || fb.score > best.score) { second = best; best = fb; }
            else if (second.frag < 0 || fb.score > second.score) { second = fb; }
        }
        out[2 * r] = best;
        out[2 * r + 1] = second;
        free(rev);
    }
    free(gp);
}

/*
 * Base qualities (section 2.2.1): "let x be the probability that the base at position i is correctly
 * sequenced.  This can be calculated by the phred score ...  The score of a match against the nucleotide at position i
 * is match x x and mismatch is mismatch x x/3."  Phred: Q = -10 log10(P(error)), so x = 1 - 10^(-Q/10).
 * The paper keeps these as floats; here they are fixed-point integers (reading 22): `scale` units per score
 * point, rounded to nearest (halves away from zero), decided in IEEE double:
 *     pmatch[i] = round(scale*match*x_i),   pmismatch[i] = round(scale*mismatch*x_i/3).
 */
void oracle_pssm_from_phred(const uint8_t *qual, int64_t n, int32_t match, int32_t mismatch, int32_t scale,
                            int32_t *pmatch, int32_t *pmismatch)
{
    for (int64_t i = 0; i < n; i++) {
        double x = 1.0 - pow(10.0, -(double)qual[i] / 10.0);
        pmatch[i] = (int32_t)llround((double)scale * (double)match * x);
        pmismatch[i] = (int32_t)llround((double)scale * (double)mismatch * x / 3.0);
    }
}

/* Position-specific score of read position i (already strand-oriented) against genome base b: "a position specific
 * scoring matrix for each read".  N on either side is a mismatch (reading 6). */
static int32_t pssm_score(uint8_t rb, uint8_t gb, int32_t pm, int32_t pmm)
{
    return (rb < 4 && rb == gb) ? pm : pmm;
}

/* First phase with a position-specific scoring matrix: oracle_map_reads with s(read[i], genome[g+i]) replaced by the
 * per-position pair (pmatch[i], pmismatch[i]).  pmatch/pmismatch are rows of `read_stride` int32 per read, indexed by
 * the position in the read as given (forward); on the reverse strand position i of the reverse-complemented read
 * carries the scores of original position m-1-i (the quality belongs to the base call). */
void oracle_map_reads_pssm(const uint8_t *genome, int64_t G, int32_t F, int32_t V,
                           const uint8_t *reads, int32_t read_stride, const int32_t *lens, int32_t n_reads,
                           const int32_t *pmatch, const int32_t *pmismatch, int32_t strands, ohit_t *out)
{
    int64_t nfrag = (G + F - 1) / F;
    int32_t max_m = 0;
    for (int32_t r = 0; r < n_reads; r++) if (lens[r] > max_m) max_m = lens[r];
    uint8_t *gp = padded_genome(genome, G, nfrag * F + max_m);
    for (int32_t r = 0; r < n_reads; r++) {
        int32_t m = lens[r];
        const uint8_t *fwd = reads + (int64_t)r * read_stride;
        const int32_t *pm = pmatch + (int64_t)r * read_stride, *pmm = pmismatch + (int64_t)r * read_stride;
        uint8_t *rev = (uint8_t *)malloc((size_t)(m > 0 ? m : 1));
        int32_t *rpm = (int32_t *)malloc(sizeof(int32_t) * (size_t)(m > 0 ? m : 1));
        int32_t *rpmm = (int32_t *)malloc(sizeof(int32_t) * (size_t)(m > 0 ? m : 1));
        reverse_complement(fwd, m, rev);
        for (int32_t i = 0; i < m; i++) { rpm[i] = pm[m - 1 - i]; rpmm[i] = pmm[m - 1 - i]; }
        int32_t Veff = (V < 0 || V > m - 1) ? m - 1 : V;
        ohit_t best = { -1, 0, 0, 0 }, second = { -1, 0, 0, 0 };
        for (int64_t f = 0; f < nfrag; f++) {
            int64_t end = f * F + F + Veff;
            ohit_t fb = { (int32_t)f, 0, -1, 0 };
            for (int32_t s = 0; s < 2; s++) {
                if (!(strands & (1 << s))) continue;
                const uint8_t *q = s ? rev : fwd;
                const int32_t *qm = s ? rpm : pm, *qmm = s ? rpmm : pmm;
                for (int32_t d = 0; d < F; d++) {
                    int64_t g = f * F + d;
                    int32_t n = (end - g < m) ? (int32_t)(end - g) : m;
                    int32_t H = 0, b = 0;
                    for (int32_t i = 0; i < n; i++) {
                        H += pssm_score(q[i], gp[g + i], qm[i], qmm[i]);
                        if (H < 0) H = 0;
                        if (H > b) b = H;
                    }
                    if (b > fb.score) { fb.score = b; fb.diag = d; fb.strand = s; }
                }
            }
            if (best.frag < 0 || fb.score > best.score) { second = best; best = fb; }
            else if (second.frag < 0 || fb.score > second.score) { second = fb; }
        }
        out[2 * r] = best;
        out[2 * r + 1] = second;
        free(rev); free(rpm); free(rpmm);
    }
    free(gp);
}

/* Second phase with the same position-specific scores ("in both phases of the program"):
 * oracle_nw_align with s(Q[i-1], W[j-1]) = pmatch/pmismatch of read position i-1 (strand-oriented as above); `gap` is
 * given in the same fixed-point units (scale*gap).  Window, recurrence, end column, traceback order and CIGAR as in
 * oracle_nw_align. */
void oracle_nw_align_pssm(const uint8_t *genome, int64_t G, int32_t F, int32_t V,
                          const uint8_t *reads, int32_t read_stride, const int32_t *lens, int32_t n_reads,
                          const ohit_t *top2, const int32_t *pmatch, const int32_t *pmismatch, int32_t gap, int32_t pad,
                          int32_t *score_out, int64_t *pos_out, uint32_t *cigar_out, int32_t cigar_stride, int32_t *ncig_out)
{
    for (int32_t r = 0; r < n_reads; r++) {
        ohit_t h = top2[2 * r];
        int32_t m = lens[r];
        if (h.frag < 0) { score_out[r] = 0; pos_out[r] = -1; ncig_out[r] = 0; continue; }
        uint8_t *q = (uint8_t *)malloc((size_t)m);
        int32_t *qm = (int32_t *)malloc(sizeof(int32_t) * (size_t)m), *qmm = (int32_t *)malloc(sizeof(int32_t) * (size_t)m);
        const int32_t *pm = pmatch + (int64_t)r * read_stride, *pmm = pmismatch + (int64_t)r * read_stride;
        if (h.strand) {
            reverse_complement(reads + (int64_t)r * read_stride, m, q);
            for (int32_t i = 0; i < m; i++) { qm[i] = pm[m - 1 - i]; qmm[i] = pmm[m - 1 - i]; }
        } else {
            memcpy(q, reads + (int64_t)r * read_stride, (size_t)m);
            for (int32_t i = 0; i < m; i++) { qm[i] = pm[i]; qmm[i] = pmm[i]; }
        }
        int32_t Veff = (V < 0 || V > m - 1) ? m - 1 : V;
        int64_t ws = (int64_t)h.frag * F - pad;           if (ws < 0) ws = 0;
        int64_t we = (int64_t)h.frag * F + F + Veff + pad; if (we > G) we = G;
        int64_t L = we - ws, cols = L + 1;
        int32_t *D = (int32_t *)malloc(sizeof(int32_t) * (size_t)(m + 1) * (size_t)cols);
        for (int64_t j = 0; j <= L; j++) D[j] = 0;
        for (int32_t i = 1; i <= m; i++) {
            D[(int64_t)i * cols] = i * gap;
            for (int64_t j = 1; j <= L; j++) {
                int32_t dg = D[(int64_t)(i - 1) * cols + j - 1] + pssm_score(q[i - 1], genome[ws + j - 1], qm[i - 1], qmm[i - 1]);
                int32_t up = D[(int64_t)(i - 1) * cols + j] + gap;
                int32_t lf = D[(int64_t)i * cols + j - 1] + gap;
                int32_t v = dg;
                if (up > v) v = up;
                if (lf > v) v = lf;
                D[(int64_t)i * cols + j] = v;
            }
        }
        int64_t jbest = 0;
        for (int64_t j = 1; j <= L; j++)
            if (D[(int64_t)m * cols + j] > D[(int64_t)m * cols + jbest]) jbest = j;
        score_out[r] = D[(int64_t)m * cols + jbest];
        uint8_t *ops = (uint8_t *)malloc((size_t)(m + L + 1));
        int64_t nops = 0;
        int32_t i = m; int64_t j = jbest;
        while (i > 0) {
            int32_t v = D[(int64_t)i * cols + j];
            if (j > 0 && D[(int64_t)(i - 1) * cols + j - 1] + pssm_score(q[i - 1], genome[ws + j - 1], qm[i - 1], qmm[i - 1]) == v) {
                ops[nops++] = 0; i--; j--;
            } else if (D[(int64_t)(i - 1) * cols + j] + gap == v) {
                ops[nops++] = 1; i--;
            } else {
                ops[nops++] = 2; j--;
            }
        }
        pos_out[r] = ws + j;
        int32_t nc = 0;
        uint32_t *cg = cigar_out + (int64_t)r * cigar_stride;
        for (int64_t k = nops - 1; k >= 0; ) {
            uint8_t op = ops[k]; uint32_t len = 0;
            while (k >= 0 && ops[k] == op) { len++; k--; }
            if (nc < cigar_stride) cg[nc] = (len << 4) | op;
            nc++;
        }
        ncig_out[r] = nc;
        free(ops); free(D); free(q); free(qm); free(qmm);
    }
}

/*
 * Repeat filter and mapping quality on the top-2 records of the first phase (next row f1).
 *   PAPER.md:57 (section 2.2.1): "it outputs the fragment number with the highest and second highest score and considers
 *   the read to be mapped if the ratio of the second best to best score is below .9".
 *   "In the MAPQ field of SAM we use the formula -100 log2 p where p is the probability of alignment being
 *   incorrect.  We define this to be the ratio of the scores of the second highest and top scoring fragments.  For
 *   MaxSSmap we consider the read mapped only if mapping quality is above -100 log2 .9 = 15.2."
 *   "we raise the MaxSSmap mapping quality threshold from the default 15.2 to 62".
 * Per record, in this order:
 *   - no best fragment (frag < 0) or best.score <= 0: the ratio is undefined -> unmapped, MAPQ 0 (reading 17);
 *   - p = second.score / best.score in double, with second.score taken as 0 when there is no second fragment (a genome
 *     of one fragment); p = 0 gives MAPQ = +infinity (nothing competes), otherwise MAPQ = -100 * log2(p) in double;
 *   - threshold < 0 selects the paper's default in its exact form, "ratio below .9", decided on the integers
 *     (10 * second < 9 * best) because the printed 15.2 is a rounded -100 log2 .9 = 15.2003 and would let a ratio of exactly .9
 *     pass; threshold >= 0 is a mapping-quality cutoff as in PAPER.md:184: mapped iff MAPQ > threshold.
 */
void oracle_mapq_filter(const void *top2_v, int32_t n_reads, double threshold, uint8_t *mapped, double *mapq)
{
    const ohit_t *top2 = (const ohit_t *)top2_v;
    for (int32_t r = 0; r < n_reads; r++) {
        ohit_t best = top2[2 * r], second = top2[2 * r + 1];
        if (best.frag < 0 || best.score <= 0) { mapped[r] = 0; mapq[r] = 0.0; continue; }
        int32_t s2 = (second.frag >= 0) ? second.score : 0;
        double p = (double)s2 / (double)best.score;
        double q = (p > 0.0) ? -100.0 * log2(p) : INFINITY;
        mapq[r] = q;
        if (threshold < 0.0) mapped[r] = (10ll * (long long)s2 < 9ll * (long long)best.score) ? 1 : 0;
        else mapped[r] = (q > threshold) ? 1 : 0;
    }
}
