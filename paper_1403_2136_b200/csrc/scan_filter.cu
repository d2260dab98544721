// Two-pass MaxSS scan, pass 1: a bounded-error fragment score for every (read, strand, fragment), at half the
// shared-memory bytes and a third of the DPX instructions per cell of the exact scan.  Pass 2 (scan_dpx_kernel with
// p.ubound set) then runs the exact scan only on the fragments that can still reach a read's top-2, so the records are
// bit-identical to the one-pass scan.
//
// Max-plus composition of two Kadane steps: with scores s1, s2 of two consecutive scored read positions
//     H2 = max(max(H + s1, 0) + s2, 0) = max(H + (s1 + s2), s2, 0).
// Pass 1 drops the middle term and samples H only after every second step:
//     G2 = max(G + a, 0),  a = s1 + s2   one LDS.32 + one VIADDMNMX.S16x2.RELU per 4 cells (two lanes x two steps)
//     Bt = max(Bt, G2)                   one VIMNMX3.S16x2 per 8 cells
// Bounds (match M > 0 > mismatch X): 0 <= H - G <= min(M, -X) at every even step (the dropped term only matters for
// (s1, s2) = (X, M) with H < -X), and an unsampled odd step lies at most -X above the next even one, hence
//     Bt <= best <= Bt + delta,   delta = min(M, -X) - X.
// The operand a depends on the read's base pair (c1, c2) and the genome pair (G[x], G[x+istep]): 16 "dibase" planes per
// tile, plus 4 planes (c1, pad) with a = s1 for the last step of an odd-length query (the loop runs the exact number of
// double steps, so no padding steps exist).  Queries holding an N (rare) are not scanned: their bound is 0xFFFF =
// "every fragment is a candidate".
#include "mss_common.cuh"

namespace {

constexpr int FQ_MAX = 32;          // queries (read x strand) per block
constexpr int NPLANE = 20;          // 4 x (4 + pad) dibase planes

struct FilterGeom { int32_t n_groups, n_splits, frags_per_split, reads_per_group; };

__device__ __forceinline__ uint32_t fpack2(int32_t lo, int32_t hi)
{
    return ((uint32_t)lo & 0xFFFFu) | ((uint32_t)hi << 16);
}

template <int K, int T>
__global__ void __launch_bounds__(T)
scan_filter_kernel(ScanParams p, FilterGeom ug, int32_t MP, int32_t ROWW, uint16_t* __restrict__ ubound)
{
    constexpr int HALF = K * T, D = 2 * K * T, NW = T / 32;
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t* planes = smem;                                   // NPLANE * ROWW
    uint32_t* roff = planes + NPLANE * ROWW;                   // FQ_MAX * MP   (one entry per double step)
    uint32_t* wres = roff + FQ_MAX * MP;                       // FQ_MAX * NW
    int32_t* qlen = (int32_t*)(wres + FQ_MAX * NW);            // FQ_MAX: double steps; 0 = not scanned
    uint32_t* cur = (uint32_t*)(qlen + FQ_MAX);                // FQ_MAX: running fragment maximum
    int32_t* forced = (int32_t*)(cur + FQ_MAX);                // FQ_MAX: 1 = bound is "candidate everywhere"

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t group = blockIdx.x % ug.n_groups, split = blockIdx.x / ug.n_groups;
    const int32_t ns = (p.strands == 3) ? 2 : 1;
    const int32_t r0 = group * ug.reads_per_group;
    const int32_t nr = min(ug.reads_per_group, p.n_reads - r0);
    const int32_t nq = nr * ns;
    const int32_t f_begin = split * ug.frags_per_split;
    const int32_t f_end = min(p.n_frag, f_begin + ug.frags_per_split);
    const int32_t istep = p.istep;

    // ---- read prep: per double step the byte offset of its dibase plane column ----------------------------------
    for (int32_t q = warp; q < nq; q += NW) {
        int32_t r = r0 + q / ns;
        int32_t strand = (ns == 2) ? (q & 1) : (p.strands == 2 ? 1 : 0);
        int32_t m = p.lens[r];
        bool ok = (m >= 1 && m <= p.max_len);
        const uint32_t* rw = p.reads + (int64_t)r * p.stride_words;
        const uint32_t* rn = p.reads_nmask ? p.reads_nmask + (int64_t)r * ((p.stride_words + 1) / 2) : nullptr;
        bool has_n = false;
        for (int32_t j = lane; j < MP; j += 32) {
            const int32_t i1 = 2 * j * istep, i2 = i1 + istep;  // the two read positions of double step j
            uint32_t plane = 0u, col = 0u;                      // past the query's last double step: never read
            if (ok && i1 < m) {
                uint32_t b1 = read_base(rw, rn, m, i1, strand);
                uint32_t b2 = (i2 < m) ? read_base(rw, rn, m, i2, strand) : 5u;     // 5 = past the end (pad)
                if (b1 == 4u || b2 == 4u) has_n = true;
                else { plane = b1 * 5u + (b2 == 5u ? 4u : b2); col = (uint32_t)i1; }
            }
            roff[q * MP + j] = (plane * (uint32_t)ROWW + col) * 4u;
        }
        has_n = __any_sync(0xffffffffu, has_n);
        if (lane == 0) {
            int32_t steps = ok ? (m + istep - 1) / istep : 0;
            qlen[q] = (ok && !has_n) ? (steps + 1) / 2 : 0;
            forced[q] = (ok && !has_n) ? 0 : 1;
        }
    }
    if (tid < FQ_MAX) cur[tid] = 0u;

    const char* my = reinterpret_cast<const char*>(planes + tid);
    const uint32_t zero = (uint32_t)p.zero;
    const int32_t tiles_per_frag = (p.F + D - 1) / D;
    const int32_t M = p.match, X = p.mismatch;

    for (int32_t f = f_begin; f < f_end; f++) {
        const int64_t fstart = (int64_t)f * p.F;
        const int64_t trunc = (p.V < 0) ? (int64_t)0x7FFFFFFFFFFFFFFFll : fstart + p.F + p.V;
        for (int32_t tile = 0; tile < tiles_per_frag; tile++) {
            const int32_t toff = tile * D;
            const int64_t g0 = fstart + toff;
            const int32_t nvalid = min(D, p.F - toff);
            __syncthreads();
            // ---- stage the tile as dibase planes ---------------------------------------------------------------
            for (int32_t x = tid; x < ROWW; x += T) {
                int64_t plo = g0 + x, phi = plo + HALF;
                uint32_t lo1 = plo < trunc ? base_at(p.gpacked, p.gnmask, plo) : 4u;
                uint32_t lo2 = plo + istep < trunc ? base_at(p.gpacked, p.gnmask, plo + istep) : 4u;
                uint32_t hi1 = phi < trunc ? base_at(p.gpacked, p.gnmask, phi) : 4u;
                uint32_t hi2 = phi + istep < trunc ? base_at(p.gpacked, p.gnmask, phi + istep) : 4u;
#pragma unroll
                for (uint32_t c1 = 0; c1 < 4; c1++) {
                    int32_t sl = lo1 == c1 ? M : X, sh = hi1 == c1 ? M : X;
#pragma unroll
                    for (uint32_t c2 = 0; c2 < 4; c2++)
                        planes[(c1 * 5 + c2) * ROWW + x] = fpack2(sl + (lo2 == c2 ? M : X), sh + (hi2 == c2 ? M : X));
                    planes[(c1 * 5 + 4) * ROWW + x] = fpack2(sl, sh);
                }
            }
            __syncthreads();

            // ---- every scanned query against the tile ----------------------------------------------------------
            for (int32_t q = 0; q < nq; q++) {
                const int32_t m2 = qlen[q];
                if (m2 == 0) { if (lane == 0) wres[q * NW + warp] = 0u; continue; }
                const uint32_t* ro = roff + q * MP;
                uint32_t H[K], B[K];
#pragma unroll
                for (int k = 0; k < K; k++) { H[k] = 0u; B[k] = 0u; }
                int32_t j0 = 0;
                for (; j0 + 4 <= m2; j0 += 4) {
                    const uint4 o = *reinterpret_cast<const uint4*>(ro + j0);
                    uint32_t Ha[K];
#pragma unroll
                    for (int k = 0; k < K; k++) Ha[k] = __viaddmax_s16x2(H[k], *reinterpret_cast<const uint32_t*>(my + o.x + k * T * 4), zero);
#pragma unroll
                    for (int k = 0; k < K; k++) H[k] = __viaddmax_s16x2(Ha[k], *reinterpret_cast<const uint32_t*>(my + o.y + k * T * 4), zero);
#pragma unroll
                    for (int k = 0; k < K; k++) B[k] = __vimax3_s16x2(B[k], Ha[k], H[k]);
#pragma unroll
                    for (int k = 0; k < K; k++) Ha[k] = __viaddmax_s16x2(H[k], *reinterpret_cast<const uint32_t*>(my + o.z + k * T * 4), zero);
#pragma unroll
                    for (int k = 0; k < K; k++) H[k] = __viaddmax_s16x2(Ha[k], *reinterpret_cast<const uint32_t*>(my + o.w + k * T * 4), zero);
#pragma unroll
                    for (int k = 0; k < K; k++) B[k] = __vimax3_s16x2(B[k], Ha[k], H[k]);
                }
                if (m2 & 2) {                                   // remainder: two double steps ...
                    const uint2 o = *reinterpret_cast<const uint2*>(ro + j0);
                    uint32_t Ha[K];
#pragma unroll
                    for (int k = 0; k < K; k++) Ha[k] = __viaddmax_s16x2(H[k], *reinterpret_cast<const uint32_t*>(my + o.x + k * T * 4), zero);
#pragma unroll
                    for (int k = 0; k < K; k++) H[k] = __viaddmax_s16x2(Ha[k], *reinterpret_cast<const uint32_t*>(my + o.y + k * T * 4), zero);
#pragma unroll
                    for (int k = 0; k < K; k++) B[k] = __vimax3_s16x2(B[k], Ha[k], H[k]);
                    j0 += 2;
                }
                if (m2 & 1) {                                   // ... and / or one
                    const uint32_t o = ro[j0];
#pragma unroll
                    for (int k = 0; k < K; k++) H[k] = __viaddmax_s16x2(H[k], *reinterpret_cast<const uint32_t*>(my + o + k * T * 4), zero);
#pragma unroll
                    for (int k = 0; k < K; k++) B[k] = __vmaxs2(B[k], H[k]);
                }
                if (nvalid < D) {                               // ragged last tile: drop foreign window starts
#pragma unroll
                    for (int k = 0; k < K; k++) {
                        int dlo = k * T + tid;
                        if (dlo >= nvalid) B[k] &= 0xFFFF0000u;
                        if (dlo + HALF >= nvalid) B[k] &= 0x0000FFFFu;
                    }
                }
                uint32_t mx = B[0];
#pragma unroll
                for (int k = 1; k < K; k++) mx = __vmaxs2(mx, B[k]);
                uint32_t W = __reduce_max_sync(0xffffffffu, max(mx & 0xFFFFu, mx >> 16));
                if (lane == 0) wres[q * NW + warp] = W;
            }
            __syncthreads();
            if (tid < nq) {
                uint32_t c = cur[tid];
                for (int w = 0; w < NW; w++) c = max(c, wres[tid * NW + w]);
                if (tile == tiles_per_frag - 1) {
                    int32_t r = r0 + tid / ns, s = tid % ns;
                    ubound[((int64_t)r * ns + s) * p.n_frag + f] = forced[tid] ? (uint16_t)0xFFFFu : (uint16_t)c;
                    c = 0u;
                }
                cur[tid] = c;
            }
        }
    }
}

struct FVariant { int K, T; };
const FVariant kFVariants[] = { {4, 256}, {4, 128}, {4, 64}, {8, 128}, {8, 256} };

struct FSmem { int32_t MP, ROWW; size_t bytes; };
FSmem filter_smem(int half, int nw, int32_t max_len, int32_t istep)
{
    FSmem s;
    int32_t steps = (max_len + istep - 1) / istep;
    s.MP = (((steps + 1) / 2) + 3) & ~3;
    int32_t MPL = (max_len + 3) & ~3;
    if (MPL < s.MP) MPL = s.MP;
    s.ROWW = (half + MPL + 3) & ~3;
    s.bytes = (size_t)(NPLANE * s.ROWW + FQ_MAX * s.MP + FQ_MAX * nw) * 4 + 3 * FQ_MAX * 4;
    return s;
}

// the tile with the least padding among those that leave room for two blocks per SM; -1 = none
thread_local int g_filter_force = -1;      // tuning hook (mss_set_scan_variant 8..12): force one pass-1 tile geometry
thread_local bool g_filter_tile_kernel = false;   // mss_set_scan_variant 8..13: this file's kernel even where the lane-per-query one applies

int pick_filter_variant(const mss_genome* g, const ScanParams& p)
{
    if (g_filter_force >= 0 && g_filter_force < 5) {
        const FVariant& v = kFVariants[g_filter_force];
        if (filter_smem(v.K * v.T, v.T / 32, p.max_len, p.istep).bytes + 2048 <= (size_t)g->max_smem_optin) return g_filter_force;
    }
    int best = -1; double best_waste = 1e30;
    for (int i = 0; i < 3; i++) {
        const FVariant& v = kFVariants[i];
        if (filter_smem(v.K * v.T, v.T / 32, p.max_len, p.istep).bytes * 2 + 4096 > (size_t)g->max_smem_optin) continue;
        int D = 2 * v.K * v.T;
        double waste = (double)((g->frag_len + D - 1) / D) * D / g->frag_len;
        if (waste < best_waste - 1e-9) { best_waste = waste; best = i; }
    }
    return best;
}

FilterGeom filter_geom(const mss_genome* g, int32_t n_reads, int32_t strands)
{
    FilterGeom ug;
    int32_t ns = strands == 3 ? 2 : 1;
    ug.reads_per_group = FQ_MAX / ns;
    ug.n_groups = (n_reads + ug.reads_per_group - 1) / ug.reads_per_group;
    if (ug.n_groups < 1) ug.n_groups = 1;
    int64_t target = (int64_t)g->sm_count * 2 * 48;            // ~48 waves of the 2 resident blocks per SM
    int64_t want = (target + ug.n_groups - 1) / ug.n_groups;
    if (want < 1) want = 1;
    if (want > g->n_frag) want = g->n_frag;
    ug.frags_per_split = (int32_t)((g->n_frag + want - 1) / want);
    ug.n_splits = (g->n_frag + ug.frags_per_split - 1) / ug.frags_per_split;
    return ug;
}

template <int K, int T>
cudaError_t launch_filter_variant(const mss_genome* g, const ScanParams& p, uint16_t* ubound, cudaStream_t st, int32_t* grid_out,
                                  int32_t* smem_out)
{
    FSmem sg = filter_smem(K * T, T / 32, p.max_len, p.istep);
    FilterGeom ug = filter_geom(g, p.n_reads, p.strands);
    cudaError_t e = cudaFuncSetAttribute(scan_filter_kernel<K, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sg.bytes);
    if (e != cudaSuccess) return e;
    int64_t blocks = (int64_t)ug.n_groups * ug.n_splits;
    scan_filter_kernel<K, T><<<(unsigned)blocks, T, sg.bytes, st>>>(p, ug, sg.MP, sg.ROWW, ubound);
    if (grid_out) *grid_out = (int32_t)blocks;
    if (smem_out) *smem_out = (int32_t)sg.bytes;
    return cudaGetLastError();
}

}  // namespace

void scan_filter_force_variant(int v, bool tile_kernel) { g_filter_force = v; g_filter_tile_kernel = tile_kernel; }

bool scan_filter_supported(const mss_genome* g, const ScanParams& p)
{
    if (g->frag_len < 256 || g->n_frag < 8) return false;       // nothing to prune
    if ((int64_t)p.max_len * p.match > 32767 || 2 * (int64_t)p.mismatch < -32768 || 2 * (int64_t)p.match > 32767) return false;
    if (!g_filter_tile_kernel && scan_filter_lq_supported(g, p)) return true;
    if (p.pssm) return false;                                   // position-specific scores: only the lane-per-query kernel bounds them
    return pick_filter_variant(g, p) >= 0;
}

int32_t scan_filter_delta(const ScanParams& p)
{
    int32_t a = p.match < -p.mismatch ? p.match : -p.mismatch;
    return a - p.mismatch;
}

cudaError_t launch_scan_filter(const mss_genome* g, const ScanParams& p, uint16_t* ubound, cudaStream_t st, int32_t* grid_out,
                               int32_t* smem_out, int32_t* tile_out, int32_t* rpb_out, int32_t* kind_out)
{
    if (!g_filter_tile_kernel && scan_filter_lq_supported(g, p))
        return launch_scan_filter_lq(g, p, ubound, st, grid_out, smem_out, tile_out, rpb_out, kind_out);
    if (kind_out) *kind_out = 1;
    int v = pick_filter_variant(g, p);
    if (v < 0) return cudaErrorInvalidConfiguration;
    if (tile_out) *tile_out = 2 * kFVariants[v].K * kFVariants[v].T;
    if (rpb_out) *rpb_out = FQ_MAX / (p.strands == 3 ? 2 : 1);
    switch (v) {
        case 0: return launch_filter_variant<4, 256>(g, p, ubound, st, grid_out, smem_out);
        case 1: return launch_filter_variant<4, 128>(g, p, ubound, st, grid_out, smem_out);
        case 2: return launch_filter_variant<4, 64>(g, p, ubound, st, grid_out, smem_out);
        case 3: return launch_filter_variant<8, 128>(g, p, ubound, st, grid_out, smem_out);
        default: return launch_filter_variant<8, 256>(g, p, ubound, st, grid_out, smem_out);
    }
}
