// a7: second stage -- Needleman-Wunsch of each read against its best region (readings 14-16).
//
// Fitting alignment with a linear gap:  D[0][j] = 0, D[i][0] = i*gap,
//     D[i][j] = max(D[i-1][j-1] + s(Q[i-1], W[j-1]), D[i-1][j] + gap, D[i][j-1] + gap),
// score = max_j D[m][j] at the smallest such j; traceback prefers diagonal, then up (I), then left (D).
//
// One warp per read, systolic over columns: lane l owns RB consecutive rows of a 32*RB-row band and works on column
// t - l at step t; the bottom value of its strip and the window base travel to lane l+1 by shuffle.  Reads longer
// than one band run band after band through a per-warp boundary row in the workspace.
//   pass 1: all L columns of the window, no storage -> score and end column j*.
//   pass 2: only the columns the optimal path can touch, [j* - W, j*] with W = m + floor((match*m - score)/|gap|) + 1
//           (a path with k deleted window bases scores at most match*m - k*|gap|), storing 2 direction bits per cell;
//           the restricted recurrence reproduces D on every cell of the optimal path, so the traceback is identical
//           (DESIGN.md section 5.4).  Lane 0 walks back and run-length encodes; the warp writes the CIGAR in read order.
#include "mss_common.cuh"

namespace {

constexpr int NW_WARPS = 4;
constexpr int NW_CH = 512;             // window bases decoded to shared memory per refill

struct NwParams {
    const uint32_t* gpacked; const uint32_t* gnmask; int64_t n_bases; int32_t F, V;
    const uint32_t* reads; const uint32_t* reads_nmask; int32_t stride_words; const int32_t* lens; int32_t n_reads, max_len;
    const mss_top2_t* hits; int32_t match, mismatch, gap, pad;
    const uint32_t* pssm; int32_t pssm_stride;  // nullable: per-position (pmatch, pmismatch) rows ("both phases")
    int32_t* score; int64_t* ref_pos; uint32_t* cigar; int32_t cigar_stride; int32_t* n_cigar;
    // workspace, per warp slot
    int32_t* bnd; int64_t bnd_stride;          // boundary row between bands
    uint32_t* tb; int64_t tb_stride;           // direction words [band][column][lane]
    uint32_t* runs; int64_t runs_stride;       // reversed run-length ops
    int32_t wmax;                              // columns reserved per band in tb
};

// One band of the systolic recurrence over window columns (c0, c0+ncols] (c0 = the column treated as column 0).
// Returns through best/jbest the running (max, smallest column) of row m when this band holds it.
template <int RB, bool TRACE>
__device__ __forceinline__ void nw_band(const NwParams& p, const uint32_t* q /*RB codes of this lane*/,
                                        const int32_t* qm /*RB match scores*/, const int32_t* qx /*RB mismatch scores*/, int32_t row0 /*rows above this lane's strip*/,
                                        bool first_band, bool last_band_store, int64_t wstart /*genome position of column c0+1*/,
                                        int32_t ncols, int32_t* bnd, uint32_t* tb_band, uint8_t* wbuf,
                                        int32_t lm, int32_t rm, bool holds_m, int32_t& best, int32_t& jbest, int32_t m)
{
    const int lane = threadIdx.x & 31;
    int32_t Dl[RB];
#pragma unroll
    for (int r = 0; r < RB; r++) Dl[r] = (row0 + r + 1) * p.gap;
    int32_t diag0 = row0 * p.gap;              // D[row0][column 0]; 0 for the very first row (row0 = 0)
    int32_t bottom = 0;
    uint32_t wb_out = 4u;
    if (holds_m && lane == lm) { best = m * p.gap; jbest = 0; }
    const int32_t steps = ncols + 31;
    for (int32_t t0 = 1; t0 <= steps; t0 += NW_CH) {
        // refill: decode window columns t0 .. t0+NW_CH-1 (only lane 0 consumes them, in order)
        __syncwarp();
        for (int32_t x = lane; x < NW_CH; x += 32) {
            int32_t col = t0 + x;
            wbuf[x] = (col <= ncols) ? (uint8_t)base_at(p.gpacked, p.gnmask, wstart + col - 1) : (uint8_t)4;
        }
        __syncwarp();
        const int32_t tend = min(steps, t0 + NW_CH - 1);
        for (int32_t t = t0; t <= tend; t++) {
            // inputs from the lane above (its outputs of the previous step)
            int32_t up_in = __shfl_up_sync(0xffffffffu, bottom, 1);
            uint32_t wb = __shfl_up_sync(0xffffffffu, wb_out, 1);
            if (lane == 0) {
                wb = wbuf[t - t0];
                up_in = first_band ? 0 : ((t <= ncols) ? bnd[t] : 0);
            }
            const int32_t j = t - lane;
            if (j >= 1 && j <= ncols) {
                int32_t up = up_in, dg = diag0;
                uint32_t dirs = 0;
#pragma unroll
                for (int r = 0; r < RB; r++) {
                    int32_t s = (q[r] == wb && wb < 4u) ? qm[r] : qx[r];   // N on either side (code 4) is a mismatch
                    int32_t a = dg + s, b = up + p.gap, c = Dl[r] + p.gap;
                    int32_t v = max(a, max(b, c));
                    if (TRACE) dirs |= (a == v ? 0u : (b == v ? 1u : 2u)) << (2 * r);
                    dg = Dl[r]; Dl[r] = v; up = v;
                }
                diag0 = up_in;
                bottom = Dl[RB - 1];
                if (TRACE) tb_band[(int64_t)(j - 1) * 32 + lane] = dirs;
                if (holds_m && lane == lm) {
                    int32_t v = Dl[0];
#pragma unroll
                    for (int r = 1; r < RB; r++) if (r == rm) v = Dl[r];
                    if (v > best) { best = v; jbest = j; }
                }
                if (last_band_store && lane == 31) bnd[j] = bottom;      // becomes the next band's top row
            }
            wb_out = wb;
        }
    }
}

template <int RB>
__global__ void __launch_bounds__(NW_WARPS * 32)
nw_kernel(NwParams p, int32_t n_slots)
{
    __shared__ uint8_t wbuf_all[NW_WARPS][NW_CH];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t slot = blockIdx.x * NW_WARPS + warp;
    if (slot >= n_slots) return;
    uint8_t* wbuf = wbuf_all[warp];
    int32_t* bnd = p.bnd + (int64_t)slot * p.bnd_stride;
    uint32_t* tb = p.tb + (int64_t)slot * p.tb_stride;
    uint32_t* runs = p.runs + (int64_t)slot * p.runs_stride;
    constexpr int BAND = 32 * RB;

    for (int32_t r = slot; r < p.n_reads; r += n_slots) {
        const mss_hit_t h = p.hits[r].best;
        const int32_t m = p.lens[r];
        if (h.frag < 0 || m < 1 || m > p.max_len) {
            if (lane == 0) { p.score[r] = 0; p.ref_pos[r] = -1; p.n_cigar[r] = 0; }
            continue;
        }
        const uint32_t* rw = p.reads + (int64_t)r * p.stride_words;
        const uint32_t* rn = p.reads_nmask ? p.reads_nmask + (int64_t)r * ((p.stride_words + 1) / 2) : nullptr;
        const uint32_t* prow = p.pssm ? p.pssm + (int64_t)r * p.pssm_stride : nullptr;
        const int32_t veff = (p.V < 0 || p.V > m - 1) ? m - 1 : p.V;
        int64_t ws = (int64_t)h.frag * p.F - p.pad; if (ws < 0) ws = 0;
        int64_t we = (int64_t)h.frag * p.F + p.F + veff + p.pad; if (we > p.n_bases) we = p.n_bases;
        const int32_t L = (int32_t)(we - ws);
        const int32_t nbands = (m + BAND - 1) / BAND;
        const int32_t bm = (m - 1) / BAND, lm = ((m - 1) % BAND) / RB, rm = (m - 1) % RB;

        // ---- pass 1: score and end column -------------------------------------------------------------------------
        int32_t best = 0, jbest = 0;
        for (int32_t b = 0; b < nbands; b++) {
            uint32_t q[RB]; int32_t qm[RB], qx[RB];
#pragma unroll
            for (int k = 0; k < RB; k++) {
                int32_t i = b * BAND + lane * RB + k;                  // 0-based read position
                q[k] = (i < m) ? read_base(rw, rn, m, i, h.strand) : 4u;
                qm[k] = p.match; qx[k] = p.mismatch;
                if (prow && i < m) {
                    uint32_t w = pssm_at(prow, m, i, h.strand);
                    qm[k] = (int32_t)(int16_t)(w & 0xFFFFu); qx[k] = (int32_t)(int16_t)(w >> 16);
                }
            }
            if (b > 0 && lane == 0) bnd[0] = b * BAND * p.gap;
            __syncwarp();
            nw_band<RB, false>(p, q, qm, qx, b * BAND + lane * RB, b == 0, b + 1 < nbands, ws, L, bnd, nullptr, wbuf,
                               lm, rm, b == bm, best, jbest, m);
            __syncwarp();
        }
        best = __shfl_sync(0xffffffffu, best, lm);
        jbest = __shfl_sync(0xffffffffu, jbest, lm);

        // ---- pass 2: the columns the optimal path can touch, with direction bits ------------------------------------
        int64_t slack = ((int64_t)p.match * m - best) / (int64_t)(-p.gap);
        int64_t Wl = (int64_t)m + slack + 1;
        if (Wl > p.wmax) Wl = p.wmax;                                  // wmax >= min(L, m + (match-mismatch)*m/|gap| + 1) always holds the path
        int32_t jlo = (int32_t)((jbest > Wl) ? (jbest - Wl) : 0);
        const int32_t Lb = jbest - jlo;
        int32_t best2 = 0, jbest2 = 0;
        for (int32_t b = 0; b < nbands; b++) {
            uint32_t q[RB]; int32_t qm[RB], qx[RB];
#pragma unroll
            for (int k = 0; k < RB; k++) {
                int32_t i = b * BAND + lane * RB + k;
                q[k] = (i < m) ? read_base(rw, rn, m, i, h.strand) : 4u;
                qm[k] = p.match; qx[k] = p.mismatch;
                if (prow && i < m) {
                    uint32_t w = pssm_at(prow, m, i, h.strand);
                    qm[k] = (int32_t)(int16_t)(w & 0xFFFFu); qx[k] = (int32_t)(int16_t)(w >> 16);
                }
            }
            if (b > 0 && lane == 0) bnd[0] = b * BAND * p.gap;
            __syncwarp();
            nw_band<RB, true>(p, q, qm, qx, b * BAND + lane * RB, b == 0, b + 1 < nbands, ws + jlo, Lb, bnd,
                              tb + (int64_t)b * p.wmax * 32, wbuf, lm, rm, b == bm, best2, jbest2, m);
            __syncwarp();
        }
        // ---- traceback (lane 0), runs collected end-to-start ---------------------------------------------------------
        int32_t nruns = 0;
        int32_t jb = Lb;
        if (lane == 0) {
            int32_t i = m;
            uint32_t cur_op = 3u, cur_len = 0;
            while (i > 0) {
                uint32_t dir;
                if (jb == 0) dir = 1u;
                else {
                    int32_t b = (i - 1) / BAND, l = ((i - 1) % BAND) / RB, k = (i - 1) % RB;
                    uint32_t w = tb[((int64_t)b * p.wmax + (jb - 1)) * 32 + l];
                    dir = (w >> (2 * k)) & 3u;
                }
                if (dir == cur_op) cur_len++;
                else {
                    if (cur_len) runs[nruns++] = (cur_len << 4) | cur_op;
                    cur_op = dir; cur_len = 1;
                }
                if (dir == 0u) { i--; jb--; } else if (dir == 1u) { i--; } else { jb--; }
            }
            if (cur_len) runs[nruns++] = (cur_len << 4) | cur_op;
            p.score[r] = best;
            p.ref_pos[r] = ws + jlo + jb;
            p.n_cigar[r] = nruns;
        }
        nruns = __shfl_sync(0xffffffffu, nruns, 0);
        __syncwarp();
        uint32_t* cg = p.cigar + (int64_t)r * p.cigar_stride;
        for (int32_t k = lane; k < nruns && k < p.cigar_stride; k += 32) cg[k] = runs[nruns - 1 - k];
        __syncwarp();
    }
}

struct NwGeom { int32_t rb, nbands, wmax, lmax, n_slots; size_t bnd_stride, tb_stride, runs_stride, total; };

NwGeom nw_geom(const mss_genome* g, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t pad)
{
    NwGeom ge;
    ge.rb = (max_len + 31) / 32;
    if (ge.rb > 8) ge.rb = 8;
    if (ge.rb < 1) ge.rb = 1;
    int band = 32 * ge.rb;
    ge.nbands = (max_len + band - 1) / band;
    int64_t lmax = (int64_t)g->frag_len + (g->overlap < 0 ? max_len - 1 : (g->overlap < max_len - 1 ? g->overlap : max_len - 1)) + 2ll * pad;
    if (lmax > g->n_bases) lmax = g->n_bases;
    ge.lmax = (int32_t)lmax;
    int64_t w = (int64_t)max_len + ((int64_t)(sc.match - sc.mismatch) * max_len) / (int64_t)(-sc.gap) + 2;
    if (w > lmax) w = lmax;
    if (w < 1) w = 1;
    ge.wmax = (int32_t)w;
    ge.bnd_stride = ((size_t)lmax + 1 + 3) / 4 * 4;
    ge.tb_stride = (size_t)ge.nbands * (size_t)ge.wmax * 32;
    ge.runs_stride = ((size_t)max_len + (size_t)ge.wmax + 4 + 3) / 4 * 4;
    size_t per_slot = (ge.bnd_stride + ge.tb_stride + ge.runs_stride) * 4;
    int64_t want = ((int64_t)n_reads + NW_WARPS - 1) / NW_WARPS * NW_WARPS;
    int64_t cap = (int64_t)g->sm_count * 12 * NW_WARPS;
    if (want > cap) want = cap;
    int64_t budget = (int64_t)(3ull << 30) / (int64_t)per_slot;           // at most ~3 GiB of scratch
    if (budget < NW_WARPS) budget = NW_WARPS;
    budget = budget / NW_WARPS * NW_WARPS;
    if (want > budget) want = budget;
    if (want < NW_WARPS) want = NW_WARPS;
    ge.n_slots = (int32_t)want;
    ge.total = per_slot * (size_t)ge.n_slots + 256;
    return ge;
}

}  // namespace

size_t nw_workspace(const mss_genome* g, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t pad)
{
    return nw_geom(g, n_reads > 0 ? n_reads : 1, max_len, sc, pad).total;
}

cudaError_t launch_nw(const mss_genome* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t stride_words,
                      const int32_t* d_lens, int32_t n_reads, int32_t max_len, const mss_top2_t* d_hits,
                      const uint32_t* d_pssm, int32_t pssm_stride,
                      mss_scoring_t sc, int32_t pad, void* ws, size_t ws_bytes, cudaStream_t st,
                      int32_t* d_score, int64_t* d_ref_pos, uint32_t* d_cigar, int32_t cigar_stride, int32_t* d_n_cigar)
{
    (void)ws_bytes;
    NwGeom ge = nw_geom(g, n_reads, max_len, sc, pad);
    NwParams p;
    p.gpacked = g->packed; p.gnmask = g->nmask; p.n_bases = g->n_bases; p.F = g->frag_len; p.V = g->overlap;
    p.reads = d_reads; p.reads_nmask = d_reads_nmask; p.stride_words = stride_words; p.lens = d_lens;
    p.n_reads = n_reads; p.max_len = max_len; p.hits = d_hits;
    p.match = sc.match; p.mismatch = sc.mismatch; p.gap = sc.gap; p.pad = pad;
    p.pssm = d_pssm; p.pssm_stride = pssm_stride;
    p.score = d_score; p.ref_pos = d_ref_pos; p.cigar = d_cigar; p.cigar_stride = cigar_stride; p.n_cigar = d_n_cigar;
    int32_t* base = (int32_t*)ws;
    p.bnd = base; p.bnd_stride = (int64_t)ge.bnd_stride;
    p.tb = (uint32_t*)(base + (size_t)ge.n_slots * ge.bnd_stride); p.tb_stride = (int64_t)ge.tb_stride;
    p.runs = p.tb + (size_t)ge.n_slots * ge.tb_stride; p.runs_stride = (int64_t)ge.runs_stride;
    p.wmax = ge.wmax;
    int blocks = ge.n_slots / NW_WARPS;
    switch (ge.rb) {
        case 1: nw_kernel<1><<<blocks, NW_WARPS * 32, 0, st>>>(p, ge.n_slots); break;
        case 2: nw_kernel<2><<<blocks, NW_WARPS * 32, 0, st>>>(p, ge.n_slots); break;
        case 3: nw_kernel<3><<<blocks, NW_WARPS * 32, 0, st>>>(p, ge.n_slots); break;
        case 4: nw_kernel<4><<<blocks, NW_WARPS * 32, 0, st>>>(p, ge.n_slots); break;
        case 5: nw_kernel<5><<<blocks, NW_WARPS * 32, 0, st>>>(p, ge.n_slots); break;
        case 6: nw_kernel<6><<<blocks, NW_WARPS * 32, 0, st>>>(p, ge.n_slots); break;
        case 7: nw_kernel<7><<<blocks, NW_WARPS * 32, 0, st>>>(p, ge.n_slots); break;
        default: nw_kernel<8><<<blocks, NW_WARPS * 32, 0, st>>>(p, ge.n_slots); break;
    }
    return cudaGetLastError();
}
