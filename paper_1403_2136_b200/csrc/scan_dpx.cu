// a1-a6: the MaxSS scan as genome-tile x read-batch blocks with packed 16-bit DPX lanes.
//
// What a block does (one work unit = a group of reads x a range of fragments):
//   once:      a1 read prep -- for every query (read, strand) a row-offset table roff[i] = base(i)*ROWW + i
//   per tile:  a2 stage the tile: D = 2*K*T window starts [g0, g0+D) of one fragment plus the m-1 look-ahead are
//              turned into 5 "score planes" in shared memory: plane[c][x] = the s16x2 pair
//              ( s(c, G[g0+x]) , s(c, G[g0+x+D/2]) ), c in {A,C,G,T,N}; N / beyond-the-window positions score mismatch
//              (PAPER.md:69 padding; readings 5, 6)
//   per query: a3 Kadane -- thread t owns K lane pairs = window starts {kT+t, kT+t+D/2}; step i is
//                  H_k = max(H_k + plane[read[i]][kT+t+i], 0)       one LDS.32 + one VIADDMNMX.S16x2.RELU per 2 cells
//                  B_k = max(B_k, H_k(i), H_k(i+1))                  one VIMNMX3.S16x2 per 4 cells
//              ("maximum scoring subsequence"; the paper's look-ahead of 16 windows, becomes
//              2K windows per thread held in registers)
//              a4 fragment max: warp REDUX max + lowest window start, one slot per (query, warp)
//   per tile:  fold the per-warp slots into the read's running fragment candidate (score desc, strand asc, diag asc);
//              at the last tile of a fragment push it into the read's top-2 (a5, strictly greater, fragments ascending)
//   at end:    a6 emit the read's top-2 (or the unit's partial top-2, merged by top2_merge_kernel)
#include <vector>
#include "mss_common.cuh"

namespace {

struct DpxUnitGeom {
    int32_t n_groups, n_splits, frags_per_split, reads_per_group;
    int32_t nq;                      // queries (read x strand) per block: NQ_MAX, fewer for long reads (tables must fit)
};

template <int K, int T>
struct Cfg {
    static constexpr int HALF = K * T;
    static constexpr int D = 2 * K * T;
    static constexpr int NW = T / 32;
};

constexpr int NQ_MAX = 32;          // most queries (read x strand) per block

__device__ __forceinline__ uint32_t pack2(int32_t lo, int32_t hi)
{
    return ((uint32_t)lo & 0xFFFFu) | ((uint32_t)hi << 16);
}

// PSSM step: both lanes of h get += eq * d (eq = 0/1 per lane, d = pmatch - pmismatch >= 0) in one IMAD on the FMA pipe
// (lanes never carry: h + d <= 32767 is checked on the host), then max(. + pmismatch, 0) on the DPX pipe.
__device__ __forceinline__ uint32_t pssm_step(uint32_t h, uint32_t eq, uint32_t d, uint32_t mm, uint32_t zero)
{
    uint32_t t;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(t) : "r"(eq), "r"(d), "r"(h));
    return __viaddmax_s16x2(t, mm, zero);
}

// PSSM = false: the two global scores are baked into the planes (the paper's "trivial match or mismatch cost").
// PSSM = true : the planes hold equality bits (1 / 0 per lane) and every step applies the query position's own
//               (pmatch, pmismatch) (base-quality position-specific scoring) as
//               H = max(H + eq*(pmatch - pmismatch) + pmismatch, 0): one extra IMAD (FMA pipe) per 2 cells.
// p.istep = 2 (MaxSSmap_fast) only changes the tables built in a1: step j reads read position 2j.
template <int K, int T, bool PSSM>
__global__ void __launch_bounds__(T)
scan_dpx_kernel(ScanParams p, DpxUnitGeom ug, int32_t MP, int32_t ROWW, mss_top2_t* __restrict__ out_partial)
{
    using C = Cfg<K, T>;
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t* planes = smem;                                   // 5 * ROWW
    uint32_t* roff = planes + 5 * ROWW;                        // nq * MP
    uint2* pq = reinterpret_cast<uint2*>(roff + ug.nq * MP);   // PSSM only: nq * MP packed (pmatch x2, pmismatch x2)
    uint32_t* wres = roff + ug.nq * MP * (PSSM ? 3 : 1);       // NQ_MAX * NW
    int32_t* qlen = (int32_t*)(wres + NQ_MAX * C::NW);         // NQ_MAX
    unsigned long long* cur = (unsigned long long*)(qlen + NQ_MAX);   // NQ_MAX (per read; 8-byte aligned by layout)
    mss_hit_t* tbest = (mss_hit_t*)(cur + NQ_MAX);             // NQ_MAX
    mss_hit_t* tsecond = tbest + NQ_MAX;                       // NQ_MAX
    int32_t* thr = (int32_t*)(tsecond + NQ_MAX);               // NQ_MAX (per read): score a fragment must exceed to matter

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t group = blockIdx.x % ug.n_groups, split = blockIdx.x / ug.n_groups;
    const int32_t ns = (p.strands == 3) ? 2 : 1;
    const int32_t r0 = group * ug.reads_per_group;
    const int32_t nr = min(ug.reads_per_group, p.n_reads - r0);
    const int32_t nq = nr * ns;
    const int32_t f_begin = split * ug.frags_per_split;
    const int32_t f_end = min(p.n_frag, f_begin + ug.frags_per_split);

    // ---- a1: read prep ------------------------------------------------------------------------------------------
    for (int32_t q = warp; q < nq; q += C::NW) {
        int32_t r = r0 + q / ns;
        int32_t strand = (ns == 2) ? (q & 1) : (p.strands == 2 ? 1 : 0);
        int32_t m = p.lens[r];
        bool ok = (m >= 1 && m <= p.max_len);
        const uint32_t* rw = p.reads + (int64_t)r * p.stride_words;
        const uint32_t* rn = p.reads_nmask ? p.reads_nmask + (int64_t)r * ((p.stride_words + 1) / 2) : nullptr;
        const uint32_t* prow = PSSM ? p.pssm + (int64_t)r * p.pssm_stride : nullptr;
        for (int32_t j = lane; j < MP; j += 32) {
            const int32_t i = j * p.istep;                      // read position scored at step j
            const bool live = ok && i < m;
            uint32_t b = live ? read_base(rw, rn, m, i, strand) : 4u;
            uint32_t col = live ? (uint32_t)i : (uint32_t)j;    // dead steps: any column of the all-mismatch plane
            roff[q * MP + j] = (b * (uint32_t)ROWW + col) * 4u; // byte offset into the planes
            if (PSSM) {
                uint32_t w = live ? pssm_at(prow, m, i, strand) : 0u;      // dead steps add 0
                int32_t mt = (int32_t)(int16_t)(w & 0xFFFFu);
                uint32_t mm = w >> 16;
                pq[q * MP + j] = make_uint2((uint32_t)(mt - (int32_t)(int16_t)mm), mm | (mm << 16));   // (pmatch - pmismatch, pmismatch x2)
            }
        }
        if (lane == 0) qlen[q] = ok ? (m + p.istep - 1) / p.istep : 0;     // number of steps
    }
    if (tid < NQ_MAX) {
        cur[tid] = 0ull;
        mss_hit_t none = { -1, 0, 0, 0 };
        tbest[tid] = none;
        tsecond[tid] = none;
        thr[tid] = -1;
    }

    const char* my = reinterpret_cast<const char*>(planes + tid);
    const uint32_t zero = (uint32_t)p.zero;                     // opaque 0: keeps ptxas from re-materialising it per use
    const int32_t tiles_per_frag = (p.F + C::D - 1) / C::D;

    // ---- two-pass scan, pass 2 (one read per block): the lower bound L2 of the read's second-best fragment score ----
    // Pass 1 left u = ubound[read][strand][f] with u <= exact <= u + delta (0xFFFF = unknown).  Two fragments score at
    // least L2 = the second largest max-over-strands u, so a fragment with u + delta < L2 lies strictly below the
    // read's second place and can never enter its top-2 (a5 replaces on strictly greater): it is skipped.
    __shared__ int32_t s_top[2 * 32];
    __shared__ int32_t s_l2;
    const uint16_t* ub0 = nullptr;
    if (p.ubound) {
        ub0 = p.ubound + (int64_t)r0 * ns * p.n_frag;
        int32_t v1 = 0, v2 = 0;
        for (int32_t f = tid; f < p.n_frag; f += T) {
            int32_t u = ub0[f];
            if (ns == 2) u = max(u, (int32_t)ub0[p.n_frag + f]);
            if (u == 0xFFFF) u = 0;                             // unknown: no information for the lower bound
            if (u > v1) { v2 = v1; v1 = u; } else if (u > v2) v2 = u;
        }
        for (int off = 16; off; off >>= 1) {                    // warp top-2 (values of distinct fragments)
            int32_t o1 = __shfl_xor_sync(0xffffffffu, v1, off), o2 = __shfl_xor_sync(0xffffffffu, v2, off);
            int32_t n1 = max(v1, o1), n2 = max(min(v1, o1), max(v2, o2));
            v1 = n1; v2 = n2;
        }
        if (lane == 0) { s_top[2 * warp] = v1; s_top[2 * warp + 1] = v2; }
        __syncthreads();
        if (tid == 0) {
            int32_t a = 0, b = 0;
            for (int w = 0; w < C::NW; w++) {
                int32_t x1 = s_top[2 * w], x2 = s_top[2 * w + 1];
                int32_t n1 = max(a, x1), n2 = max(min(a, x1), max(b, x2));
                a = n1; b = n2;
            }
            s_l2 = b;
        }
        __syncthreads();
    }
    const int32_t l2 = p.ubound ? s_l2 : 0;

    for (int32_t f = f_begin; f < f_end; f++) {
        uint32_t skipq = 0u;                                    // pass 2: strands of this fragment that cannot matter
        if (ub0) {                                              // block-uniform: every thread reads the same two values
            int32_t u0 = ub0[f], u1 = (ns == 2) ? (int32_t)ub0[p.n_frag + f] : 0;
            int32_t u = max(u0, u1);
            if (u != 0xFFFF && u + p.delta < l2) continue;
            // a strand whose own bound stays below L2 scores below the read's second place: whatever it would report
            // cannot be the score that puts this fragment into the top-2, so the other strand alone represents it
            if (ns == 2 && u != 0xFFFF) {
                if (u0 + p.delta < l2) skipq |= 1u;
                if (u1 + p.delta < l2) skipq |= 2u;
            }
        }
        const int64_t fstart = (int64_t)f * p.F;
        const int64_t trunc = (p.V < 0) ? (int64_t)0x7FFFFFFFFFFFFFFFll : fstart + p.F + p.V;   // positions >= trunc are not readable
        for (int32_t tile = 0; tile < tiles_per_frag; tile++) {
            const int32_t toff = tile * C::D;
            const int64_t g0 = fstart + toff;
            const int32_t nvalid = min(C::D, p.F - toff);
            __syncthreads();                                    // previous tile fully scanned and folded
            // ---- a2: stage the tile as score planes ------------------------------------------------------------
            for (int32_t x = tid; x < ROWW; x += T) {
                int64_t plo = g0 + x, phi = plo + C::HALF;
                uint32_t lo = plo < trunc ? base_at(p.gpacked, p.gnmask, plo) : 4u;
                uint32_t hi = phi < trunc ? base_at(p.gpacked, p.gnmask, phi) : 4u;
                const int32_t eqv = PSSM ? 1 : p.match, nev = PSSM ? 0 : p.mismatch;
#pragma unroll
                for (uint32_t c = 0; c < 4; c++)
                    planes[c * ROWW + x] = pack2(lo == c ? eqv : nev, hi == c ? eqv : nev);
                planes[4 * ROWW + x] = pack2(nev, nev);
            }
            __syncthreads();

            // ---- a3/a4: every query against the tile -----------------------------------------------------------
            for (int32_t q = 0; q < nq; q++) {
                const int32_t m = qlen[q];
                if (m == 0 || ((skipq >> q) & 1u)) { if (lane == 0) wres[q * C::NW + warp] = 0u; continue; }
                const int32_t need = thr[q >> (ns - 1)];       // the read's current second-best score (or -1)
                const uint32_t* ro = roff + q * MP;
                uint32_t H[K], B[K];
#pragma unroll
                for (int k = 0; k < K; k++) { H[k] = 0u; B[k] = 0u; }
                for (int32_t i0 = 0; i0 < m; i0 += 4) {
                    const uint4 o = *reinterpret_cast<const uint4*>(ro + i0);
                    uint32_t Ha[K];
                    if (!PSSM) {
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
                    } else {
                        const uint4 s01 = *reinterpret_cast<const uint4*>(pq + q * MP + i0);        // (d0, mm0, d1, mm1)
                        const uint4 s23 = *reinterpret_cast<const uint4*>(pq + q * MP + i0 + 2);
#pragma unroll
                        for (int k = 0; k < K; k++)
                            Ha[k] = pssm_step(H[k], *reinterpret_cast<const uint32_t*>(my + o.x + k * T * 4), s01.x, s01.y, zero);
#pragma unroll
                        for (int k = 0; k < K; k++)
                            H[k] = pssm_step(Ha[k], *reinterpret_cast<const uint32_t*>(my + o.y + k * T * 4), s01.z, s01.w, zero);
#pragma unroll
                        for (int k = 0; k < K; k++) B[k] = __vimax3_s16x2(B[k], Ha[k], H[k]);
#pragma unroll
                        for (int k = 0; k < K; k++)
                            Ha[k] = pssm_step(H[k], *reinterpret_cast<const uint32_t*>(my + o.z + k * T * 4), s23.x, s23.y, zero);
#pragma unroll
                        for (int k = 0; k < K; k++)
                            H[k] = pssm_step(Ha[k], *reinterpret_cast<const uint32_t*>(my + o.w + k * T * 4), s23.z, s23.w, zero);
#pragma unroll
                        for (int k = 0; k < K; k++) B[k] = __vimax3_s16x2(B[k], Ha[k], H[k]);
                    }
                }
                // a4: warp max and its lowest window start
                if (nvalid < C::D) {                            // ragged last tile of a fragment: drop foreign window starts
#pragma unroll
                    for (int k = 0; k < K; k++) {
                        int dlo = k * T + tid;
                        if (dlo >= nvalid) B[k] &= 0xFFFF0000u;
                        if (dlo + C::HALF >= nvalid) B[k] &= 0x0000FFFFu;
                    }
                }
                uint32_t mx = B[0];
#pragma unroll
                for (int k = 1; k < K; k++) mx = __vmaxs2(mx, B[k]);
                uint32_t M = max(mx & 0xFFFFu, mx >> 16);
                uint32_t W = __reduce_max_sync(0xffffffffu, M);
                // a5 replaces only on strictly greater and fragments ascend: a fragment that does not beat the read's
                // current second place can never enter the top-2, so its window start is not needed (slot 0 = no report)
                if ((int32_t)W <= need) { if (lane == 0) wres[q * C::NW + warp] = 0u; continue; }
                uint32_t d = 0xFFFFu;
                if (M == W) {
#pragma unroll
                    for (int k = K - 1; k >= 0; k--) if ((B[k] >> 16) == W) d = (uint32_t)(k * T + tid + C::HALF);
#pragma unroll
                    for (int k = K - 1; k >= 0; k--) if ((B[k] & 0xFFFFu) == W) d = (uint32_t)(k * T + tid);
                }
                d = __reduce_min_sync(0xffffffffu, d);
                if (lane == 0) wres[q * C::NW + warp] = (W << 16) | (0xFFFFu - d);
            }
            __syncthreads();
            // ---- fold into the running fragment candidate; a5 top-2 at the fragment's last tile ------------------
            if (tid < nr) {
                unsigned long long c = cur[tid];
                for (int32_t s = 0; s < ns; s++) {
                    int32_t q = tid * ns + s;
                    if (qlen[q] == 0) continue;
                    uint32_t best = 0u;
                    for (int w = 0; w < C::NW; w++) best = max(best, wres[q * C::NW + w]);
                    if (best == 0u) continue;                   // no warp reported (a report always has a non-zero low half)
                    int32_t strand = (ns == 2) ? s : (p.strands == 2 ? 1 : 0);
                    unsigned long long k64 = frag_key((int32_t)(best >> 16), strand, toff + (int32_t)(0xFFFFu - (best & 0xFFFFu)));
                    c = k64 > c ? k64 : c;
                }
                if (tile == tiles_per_frag - 1) {
                    if (c != 0ull) {
                        mss_hit_t h; h.frag = f;
                        frag_key_unpack(c, h.score, h.strand, h.diag);
                        mss_hit_t b = tbest[tid], s2 = tsecond[tid];
                        top2_push(b, s2, h);
                        tbest[tid] = b; tsecond[tid] = s2;
                        thr[tid] = s2.frag >= 0 ? s2.score : -1;
                    }
                    c = 0ull;
                }
                cur[tid] = c;
            }
        }
    }
    __syncthreads();
    if (tid < nr) {
        mss_top2_t o; o.best = tbest[tid]; o.second = tsecond[tid];
        out_partial[(int64_t)split * p.n_reads + r0 + tid] = o;
    }
}

__global__ void top2_merge_kernel(const mss_top2_t* __restrict__ partial, int32_t n_splits, int32_t n_reads,
                                  mss_top2_t* __restrict__ out)
{
    int32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_reads) return;
    mss_hit_t none = { -1, 0, 0, 0 };
    mss_hit_t best = none, second = none;
    for (int32_t s = 0; s < n_splits; s++) {
        mss_top2_t t = partial[(int64_t)s * n_reads + r];
        top2_merge(best, second, t.best);
        top2_merge(best, second, t.second);
    }
    out[r].best = best;
    out[r].second = second;
}

DpxUnitGeom unit_geom(const mss_genome* g, int32_t n_reads, int32_t strands, int32_t nq)
{
    DpxUnitGeom ug;
    int32_t ns = strands == 3 ? 2 : 1;
    ug.nq = nq;
    ug.reads_per_group = nq / ns;
    ug.n_groups = (n_reads + ug.reads_per_group - 1) / ug.reads_per_group;
    if (ug.n_groups < 1) ug.n_groups = 1;
    // blocks are long (a group of reads against a whole range of fragments): aim for >= ~48 waves of 3 resident blocks
    // per SM so that the ragged end of the grid costs about 1 % (measured: 14 waves left ~4 % of the SMs' time idle)
    int64_t target = (int64_t)g->sm_count * 3 * 48;
    int64_t want = (target + ug.n_groups - 1) / ug.n_groups;
    if (want < 1) want = 1;
    if (want > g->n_frag) want = g->n_frag;
    if (want > 4096) want = 4096;
    ug.frags_per_split = (int32_t)((g->n_frag + want - 1) / want);
    ug.n_splits = (g->n_frag + ug.frags_per_split - 1) / ug.frags_per_split;
    return ug;
}

struct Variant { int id, K, T; };
const Variant kVariants[] = { {2, 8, 256}, {3, 8, 128}, {4, 8, 64}, {5, 4, 256}, {6, 16, 128} };

// shared-memory geometry: MP = steps per query rounded to 4 (table rows), ROWW = plane columns (tile half + read length)
struct SmemGeom { int32_t MP, ROWW; size_t bytes; };
SmemGeom smem_geom(int half, int nw, int32_t max_len, int32_t istep, bool pssm, int32_t nq)
{
    SmemGeom s;
    int32_t steps = (max_len + istep - 1) / istep;
    s.MP = (steps + 3) & ~3;
    int32_t MPL = (max_len + 3) & ~3;
    if (MPL < s.MP) MPL = s.MP;
    s.ROWW = (half + MPL + 3) & ~3;
    s.bytes = (size_t)(5 * s.ROWW + nq * s.MP * (pssm ? 3 : 1) + NQ_MAX * nw) * 4 + NQ_MAX * 4 + NQ_MAX * 8
            + 2 * NQ_MAX * sizeof(mss_hit_t) + NQ_MAX * 4;
    return s;
}

template <int K, int T, bool PSSM>
cudaError_t launch_variant2(const mss_genome* g, const ScanParams& p, const DpxUnitGeom& ug, mss_top2_t* partial,
                            cudaStream_t st, mss_launch_info_t* info, int id)
{
    using C = Cfg<K, T>;
    SmemGeom sg = smem_geom(C::HALF, C::NW, p.max_len, p.istep, PSSM, ug.nq);
    int32_t MP = sg.MP, ROWW = sg.ROWW;
    size_t smem = sg.bytes;
    if (smem > (size_t)g->max_smem_optin) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(scan_dpx_kernel<K, T, PSSM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int64_t blocks = (int64_t)ug.n_groups * ug.n_splits;
    scan_dpx_kernel<K, T, PSSM><<<(unsigned)blocks, T, smem, st>>>(p, ug, MP, ROWW, partial);
    if (info) {
        info->variant = id; info->grid = (int32_t)blocks; info->block = T; info->smem_bytes = (int32_t)smem;
        info->reads_per_block = ug.reads_per_group; info->tile_diagonals = C::D; info->launches = 2; info->pass1_kernel = 0;
    }
    return cudaGetLastError();
}

template <int K, int T>
cudaError_t launch_variant(const mss_genome* g, const ScanParams& p, const DpxUnitGeom& ug, mss_top2_t* partial,
                           cudaStream_t st, mss_launch_info_t* info, int id)
{
    return p.pssm ? launch_variant2<K, T, true>(g, p, ug, partial, st, info, id)
                  : launch_variant2<K, T, false>(g, p, ug, partial, st, info, id);
}

bool variant_fits(const mss_genome* g, const ScanParams& p, const Variant& v, int32_t nq)
{
    return smem_geom(v.K * v.T, v.T / 32, p.max_len, p.istep, p.pssm != nullptr, nq).bytes <= (size_t)g->max_smem_optin;
}

// queries per block: as many as the shared memory allows next to the smallest tile (long reads get fewer; 0 = none fits)
int32_t pick_nq(const mss_genome* g, const ScanParams& p)
{
    for (int32_t nq = NQ_MAX; nq >= 2; nq >>= 1)
        if (smem_geom(512, 2, p.max_len, p.istep, p.pssm != nullptr, nq).bytes + 32 * 1024 <= (size_t)g->max_smem_optin) return nq;
    return 0;
}

int pick_variant(const mss_genome* g, const ScanParams& p, int requested, int32_t nq)
{
    for (const Variant& v : kVariants) if (v.id == requested && variant_fits(g, p, v, nq)) return requested;
    // automatic: among the tiles whose shared memory fits, the one with the least padding waste (larger tiles on ties)
    int best = 4; double best_waste = 1e30;
    for (const Variant& v : kVariants) {
        if (v.id > 4 || !variant_fits(g, p, v, nq)) continue;        // 5, 6 are tuning variants, never automatic
        int D = 2 * v.K * v.T;
        double waste = (double)((g->frag_len + D - 1) / D) * D / g->frag_len;
        if (waste < best_waste - 1e-9) { best_waste = waste; best = v.id; }
    }
    return best;
}

}  // namespace

bool scan_dpx_supported(const mss_genome* g, const ScanParams& p)
{
    if (g->frag_len < 256) return false;                        // tiles would be mostly padding: generic kernel
    if ((int64_t)p.max_len * p.match > 32767 || p.mismatch < -32768) return false;
    // PSSM lanes hold H + (pmatch - pmismatch) before the mismatch is added back: keep that inside int16 too
    if (p.pssm && (int64_t)p.max_len * p.match + ((int64_t)p.match - p.mismatch) > 32767) return false;
    return pick_nq(g, p) >= 2;
}

size_t scan_dpx_workspace(const mss_genome* g, int32_t n_reads, int32_t max_len, int32_t strands)
{
    (void)max_len;
    int32_t n = n_reads > 0 ? n_reads : 1, most = 1;
    for (int32_t nq = NQ_MAX; nq >= 2; nq >>= 1) {               // the split count depends on the queries per block
        int32_t sp = unit_geom(g, n, strands, nq).n_splits;
        if (sp > most) most = sp;
    }
    return (size_t)most * (size_t)n * sizeof(mss_top2_t) + 256;
}

cudaError_t launch_scan_dpx(const mss_genome* g, const ScanParams& p, void* ws, size_t ws_bytes,
                            mss_top2_t* d_out, cudaStream_t st, mss_launch_info_t* info, int variant)
{
    (void)ws_bytes;
    int32_t nq = pick_nq(g, p);
    if (nq < 2) return cudaErrorInvalidConfiguration;
    DpxUnitGeom ug = unit_geom(g, p.n_reads, p.strands, nq);
    mss_top2_t* partial = (mss_top2_t*)ws;
    int id = pick_variant(g, p, variant, nq);
    cudaError_t e;
    switch (id) {
        case 3: e = launch_variant<8, 128>(g, p, ug, partial, st, info, id); break;
        case 4: e = launch_variant<8, 64>(g, p, ug, partial, st, info, id); break;
        case 5: e = launch_variant<4, 256>(g, p, ug, partial, st, info, id); break;
        case 6: e = launch_variant<16, 128>(g, p, ug, partial, st, info, id); break;
        default: e = launch_variant<8, 256>(g, p, ug, partial, st, info, 2); break;
    }
    if (e != cudaSuccess) return e;
    top2_merge_kernel<<<(p.n_reads + 255) / 256, 256, 0, st>>>(partial, ug.n_splits, p.n_reads, d_out);
    return cudaGetLastError();
}

// ---- two-pass scan: bounded-error pass 1 (scan_filter.cu), exact pass 2 on the candidate fragments ----
namespace {
// optional CUDA-event timing of the two passes on the launching stream (mss_set_pass_timing / mss_get_pass_times)
thread_local bool t_time_passes = false;
thread_local std::vector<cudaEvent_t>* t_events = nullptr;      // 3 per chunk: before pass 1, between, after pass 2
thread_local int t_events_used = 0;

cudaEvent_t next_event()
{
    if (!t_events) t_events = new std::vector<cudaEvent_t>();
    if (t_events_used == (int)t_events->size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
        t_events->push_back(e);
    }
    return (*t_events)[t_events_used++];
}

thread_local int64_t g_bounds_bytes = 256ll << 20;   // bounds produced per chunk of reads (mss_set_two_pass_chunk_bytes: tests use small values)

int32_t two_pass_chunk(const mss_genome* g, int32_t n_reads, int32_t strands)
{
    int64_t per_read = (int64_t)(strands == 3 ? 2 : 1) * g->n_frag * 2;         // bytes of bounds per read
    int64_t c = g_bounds_bytes / per_read;
    if (c < 1) c = 1;
    if (c > n_reads) c = n_reads;
    if (c < 1) c = 1;
    return (int32_t)c;
}
}  // namespace

size_t scan_two_pass_workspace(const mss_genome* g, int32_t n_reads, int32_t strands)
{
    int32_t n = n_reads > 0 ? n_reads : 1;
    return (size_t)two_pass_chunk(g, n, strands) * (size_t)(strands == 3 ? 2 : 1) * (size_t)g->n_frag * 2 + 256;
}

cudaError_t launch_scan_two_pass(const mss_genome* g, const ScanParams& p0, void* ws, size_t ws_bytes,
                                 mss_top2_t* d_out, cudaStream_t st, mss_launch_info_t* info)
{
    (void)ws_bytes;
    const int32_t ns = p0.strands == 3 ? 2 : 1;
    // chunks of equal size (whole 64-read blocks) rather than full chunks and a small rest: every launch then fills the GPU
    int32_t chunk = two_pass_chunk(g, p0.n_reads, p0.strands);
    if (chunk < p0.n_reads) {
        const int32_t n_chunks = (p0.n_reads + chunk - 1) / chunk;
        int32_t even = ((p0.n_reads + n_chunks - 1) / n_chunks + 63) & ~63;
        if (even < chunk) chunk = even;
    }
    uint16_t* ubound = (uint16_t*)ws;
    int launches = 0;
    int32_t fgrid = 0, fsmem = 0, ftile = 0, frpb = 0, fkind = 0;
    t_events_used = 0;
    for (int32_t c0 = 0; c0 < p0.n_reads; c0 += chunk) {
        cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev2 = nullptr;
        cudaError_t e;
        if (t_time_passes) {
            ev0 = next_event(); ev1 = next_event(); ev2 = next_event();
            if (!ev0 || !ev1 || !ev2) { t_events_used = 0; return cudaErrorMemoryAllocation; }
            if ((e = cudaEventRecord(ev0, st)) != cudaSuccess) { t_events_used = 0; return e; }
        }
        ScanParams p = p0;
        p.n_reads = p0.n_reads - c0 < chunk ? p0.n_reads - c0 : chunk;
        p.reads = p0.reads + (int64_t)c0 * p0.stride_words;
        p.reads_nmask = p0.reads_nmask ? p0.reads_nmask + (int64_t)c0 * ((p0.stride_words + 1) / 2) : nullptr;
        p.lens = p0.lens + c0;
        p.pssm = p0.pssm ? p0.pssm + (int64_t)c0 * p0.pssm_stride : nullptr;       // the chunk's rows of the base-quality table
        p.ubound = nullptr;
        e = launch_scan_filter(g, p, ubound, st, &fgrid, &fsmem, &ftile, &frpb, &fkind);
        if (e != cudaSuccess) return e;
        if (ev1 && (e = cudaEventRecord(ev1, st)) != cudaSuccess) { t_events_used = 0; return e; }
        // pass 2: one read per block, every fragment range in one block (the bounds row decides what is scanned)
        p.ubound = ubound;
        p.delta = scan_filter_delta(p);
        DpxUnitGeom ug;
        ug.nq = ns; ug.reads_per_group = 1; ug.n_groups = p.n_reads; ug.n_splits = 1; ug.frags_per_split = g->n_frag;
        int id = pick_variant(g, p, 0, ns);
        mss_top2_t* out = d_out + c0;
        switch (id) {
            case 3: e = launch_variant<8, 128>(g, p, ug, out, st, nullptr, id); break;
            case 4: e = launch_variant<8, 64>(g, p, ug, out, st, nullptr, id); break;
            default: e = launch_variant<8, 256>(g, p, ug, out, st, nullptr, 2); break;
        }
        if (e != cudaSuccess) return e;
        if (ev2 && (e = cudaEventRecord(ev2, st)) != cudaSuccess) { t_events_used = 0; return e; }
        launches += 2;
    }
    if (info) {
        info->variant = 7; info->grid = fgrid; info->block = 0; info->smem_bytes = fsmem;
        info->reads_per_block = frpb; info->tile_diagonals = ftile; info->launches = launches; info->pass1_kernel = fkind;
    }
    return cudaSuccess;
}

void scan_set_two_pass_chunk_bytes(int64_t bytes) { g_bounds_bytes = bytes < 1 ? (256ll << 20) : bytes; }

void scan_set_pass_timing(bool on)
{
    t_time_passes = on;
    if (!on) {                                                  // the events live only while timing is on
        t_events_used = 0;
        if (t_events) { for (cudaEvent_t ev : *t_events) cudaEventDestroy(ev); delete t_events; t_events = nullptr; }
    }
}

// sums over the chunks of the last two-pass call on this thread; synchronises on its last event
cudaError_t scan_get_pass_times(float* pass1_ms, float* pass2_ms)
{
    *pass1_ms = 0.f; *pass2_ms = 0.f;
    if (!t_events || t_events_used < 3) return cudaSuccess;
    cudaError_t e = cudaEventSynchronize((*t_events)[t_events_used - 1]);
    for (int i = 0; e == cudaSuccess && i + 2 < t_events_used; i += 3) {
        float a = 0.f, b = 0.f;
        e = cudaEventElapsedTime(&a, (*t_events)[i], (*t_events)[i + 1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&b, (*t_events)[i + 1], (*t_events)[i + 2]);
        *pass1_ms += a; *pass2_ms += b;
    }
    return e;
}
