// Two-pass MaxSS scan, pass 1, lane-per-query layout: the same bounded-error double-step recurrence as
// scan_filter.cu (G2 = max(G + s1 + s2, 0) sampled every second scored read position; bounds
// Bt <= best <= Bt + delta), with the roles of the warp lanes turned round:
//
//   scan_filter_kernel     lane <-> window start; the query is block-uniform, so the plane offset of every double step is
//                          a broadcast LDS.128 from a per-query table (one shared-memory wavefront in eight) and the
//                          fragment maximum of a query needs a warp REDUX per (query, tile, warp)
//   scan_filter_lq_kernel  lane <-> query (32 queries = 16 reads x 2 strands per warp); the window start is warp-uniform.
//                          A thread keeps its own query's plane offsets IN REGISTERS for the whole kernel (one per double
//                          step, or two 16-bit offsets per register for long reads), so a double step of a chain is one
//                          shared-memory load and one add-max-relu (+ half a 3-input max): no offset loads, no address
//                          arithmetic, and the maximum over window starts is a per-thread running max: no REDUX.
//
// Shared-memory access: the 32 lanes of a warp read the same column of up to 21 different planes.  The plane stride is
// 1 (mod 32) words, so plane p, word c lies in bank (p + c) mod 32: lanes on different planes hit different banks, lanes
// on the same plane read the same word (broadcast) -- one wavefront per LDS.32.
//
// A warp walks its share of the tile's columns in groups of K = 8 adjacent columns (8 independent chains per thread, each
// a packed pair of window starts x and x + HALF); the group base is warp-uniform.
//
// Arithmetic of the chains (template MODE; all three give the same integers, tests compare them):
//   LQ_S16   planes hold packed int16 pairs; step = VIADDMNMX.S16x2.RELU (ALU pipe), max = VIMNMX3.S16x2 (ALU pipe).
//   LQ_F16   planes hold the same integers as fp16 pairs (exact: every value is an integer of magnitude <= 2048); step =
//            HFMA2.RELU (H * 1 + a, FMA pipe), max = VIMNMX3.S16x2 on the fp16 bit patterns (non-negative fp16 values
//            order like integers).  The ALU pipe, which the integer form loads to 75 %, only carries the max.
//   LQ_F8    planes hold e5m2 bytes (= the high byte of the fp16 value; the scores of the default 5/-4 scoring and of
//            any scoring whose sums have <= 3 significant bits are exact), four per word = two adjacent columns x two
//            window starts: one LDS.32 feeds two chains, a PRMT per chain widens a byte pair to fp16x2, then as LQ_F16.
//            Half the shared-memory wavefronts per cell.
//   LQ_PSSM  base-quality scoring: every query position has its own (pmatch, pmismatch), so a double step has
//            four possible operands T[p], p = match pattern of its two positions.  The planes are query-independent as
//            before but hold, per column and window start, the PRMT SELECTOR of the pattern (byte (2p+1)<<4 | 2p); a
//            thread loads its own query's T and plane offset of the double step (one LDS.128 from a per-query table,
//            shared by its 8 chains: the offsets need no registers, so one instance serves every read length) and one
//            PRMT(T.lo, T.hi, selector) per chain yields the packed int16 operand pair; then VIADDMNMX.S16x2.RELU /
//            VIMNMX3.S16x2 as LQ_S16 (scores reach scale * match * m: no fp16).  Bound: delta = min(PM, -PMM) - PMM
//            with PM / PMM the table's largest pmatch / most negative pmismatch.
#include <cuda_fp16.h>
#include "mss_common.cuh"

namespace {

constexpr int LQ_NW = 8;            // warps per block
#ifndef LQ_K_CHAINS
#define LQ_K_CHAINS 8
#endif
#ifndef LQ_BLOCKS_PER_SM
#define LQ_BLOCKS_PER_SM 2
#endif
constexpr int LQ_K = LQ_K_CHAINS;   // adjacent columns (chains) per thread and column group
// planes of a tile: (c1, c2) -> c1*4 + c2; (c1, pad) -> 16 + c1 (last step of an odd-length query); 20 = all zero (padding
// steps).  Blocks whose reads hold an N ("N" scores mismatch against everything, reading 6) add ten more:
// (c1, N) -> 21 + c1, (N, c2) -> 25 + c2, (N, N) -> 29, (N, pad) -> 30, and take a smaller tile to make room for them.
constexpr int LQ_NPL = 21;
constexpr int LQ_NPL_N = 31;
constexpr int LQ_ZERO_PLANE = 20;
constexpr int LQ_MAX_QSETS = 4;
enum { LQ_S16 = 0, LQ_F16 = 1, LQ_F8 = 2, LQ_PSSM = 3 };
constexpr int LQ_TABLE = 8;         // host side: flag on the arithmetic = plane offsets from the shared-memory table
constexpr int LQ_K16 = 16;          // host side: flag = the 16-chain instances (short reads)
#ifndef LQ_K16_UP_TO_NJ
#define LQ_K16_UP_TO_NJ 38          // reads of at most this many double steps (76 scored positions) take the 16-chain instances
#endif
#ifndef LQ_TABLE_FROM_NJ
#define LQ_TABLE_FROM_NJ 76         // reads of more double steps than this (> 152 scored positions) take the table-driven instance
#endif

struct LqTile {
    int32_t HALF, ROWW, NG;         // tile = 2*HALF window starts; plane stride (words); column groups per warp and tile
    int32_t COLS;                   // columns staged per tile (HALF + look-ahead)
    int32_t NRAW;                   // packed genome words a tile reads (even)
};
struct LqGeom {
    int32_t n_groups, n_splits, frags_per_split, reads_per_group;
    int32_t qsets;                  // query sets (of 32 lanes) per block: 1, 2 or 4; a set is scanned by NW / qsets warps
    LqTile a;                       // blocks without an N in their reads: 21 planes
    LqTile b;                       // blocks with one: 31 planes, smaller tile (HALF = 0: none fits, such reads stay unbounded)
    int32_t tstride;                // PSSM: entries of a thread's double-step table (odd, >= the double steps of the longest read + 1)
};

__device__ __forceinline__ void lq_cp_async4(void* smem_dst, const void* gmem_src)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"(d), "l"(gmem_src) : "memory");
}

// PRMT with a register selector whose nibbles are all < 8 (__byte_perm would mask it with 0x7777 first: one LOP3 per use)
__device__ __forceinline__ uint32_t lq_prmt(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}

// x >> 16 on the FMA pipe (IMAD.HI by 2^16): the PSSM form is bound by the ALU pipe, where SHF would go
__device__ __forceinline__ uint32_t lq_hi16(uint32_t x)
{
    uint32_t d;
    asm("mul.hi.u32 %0, %1, 65536;" : "=r"(d) : "r"(x));
    return d;
}

template <int MODE>
__device__ __forceinline__ uint32_t lq_enc(int32_t v)            // one lane's operand: int16, or fp16 bits of the integer
{
    if (MODE == LQ_S16 || MODE == LQ_PSSM) return (uint32_t)v & 0xFFFFu;
    return (uint32_t)__half_as_ushort(__int2half_rn(v));
}

// NJ     = most double steps of a query this instantiation holds in registers (even); 0 = none: the plane offsets of a
//          query come from a shared-memory table, one 8-byte entry (two offsets) per pair of double steps, read by one
//          LDS.64 per pair and shared by the thread's 8 chains (any read length the table leaves room for; no padding
//          steps beyond the pair; ~50 registers fewer)
// PACKED = two 16-bit word offsets per register (long reads) instead of one byte offset per register
// KC     = chains per thread and column group (8; 16 for the short-read instances, whose few offset registers leave room: the
//          per-group start-up and the per-double-step address are shared by twice as many cells)
template <int NJ, bool PACKED, int MODE, int KC = LQ_K>
__global__ void __launch_bounds__(32 * LQ_NW, LQ_BLOCKS_PER_SM)
scan_filter_lq_kernel(ScanParams p, LqGeom ug, uint16_t* __restrict__ ubound)
{
    constexpr int K = KC, NW = LQ_NW, T = 32 * NW;
    constexpr bool TABLE = (NJ == 0);
    constexpr int NREG = TABLE ? 1 : (PACKED ? NJ / 2 : NJ);
    constexpr bool BYTEP = (MODE == LQ_F8 || MODE == LQ_PSSM);   // planes hold one byte per (column, window start): two columns per word
    // PSSM: a query's table of (operands, plane offset) per double step: ug.tstride 16-byte entries (odd: conflict-free LDS.128)
    // TABLE: a query's table of offset pairs: ug.tstride 8-byte entries (odd: conflict-free LDS.64)
    const int32_t TABW = (MODE == LQ_PSSM) ? 4 * ug.tstride : (TABLE ? 2 * ug.tstride : 0);
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t* wres = smem;                                      // NW * 32: per (warp, lane) tile maximum
    int32_t* qnj = (int32_t*)(wres + NW * 32);                  // 32 * qsets: double steps of a query; 0 = not scanned
    int32_t* qm = qnj + 32 * LQ_MAX_QSETS;                      // 32 * qsets: read length
    uint32_t* tab = (uint32_t*)(qm + 32 * LQ_MAX_QSETS);        // PSSM: 32 * qsets * TABW words, one table per query
    uint32_t* planes = tab + 32 * ug.qsets * TABW;              // NPL * ROWW (the tile geometry is chosen below)
    uint8_t* sq = reinterpret_cast<uint8_t*>(planes);           // prologue only: strand-oriented base codes, row = query

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t group = blockIdx.x % ug.n_groups, split = blockIdx.x / ug.n_groups;
    const int32_t ns = (p.strands == 3) ? 2 : 1;
    const int32_t r0 = group * ug.reads_per_group;
    const int32_t nr = min(ug.reads_per_group, p.n_reads - r0);
    const int32_t nq = nr * ns;
    const int32_t f_begin = split * ug.frags_per_split;
    const int32_t f_end = min(p.n_frag, f_begin + ug.frags_per_split);
    const int32_t istep = p.istep;
    const int32_t wps = NW / ug.qsets;                          // warps per query set
    const int32_t set = warp / wps, ws = warp % wps;
    const int32_t sq_stride = (p.max_len + 3) & ~3;

    // ---- a1 read prep, step 1: strand-oriented base codes of every query of the block (bytes; 4 = N) -----------------
    bool any_n = false;
    for (int32_t q = warp; q < 32 * ug.qsets; q += NW) {
        int32_t njq = 0, m = 0;
        if (q < nq) {
            const int32_t r = r0 + q / ns;
            const int32_t strand = (ns == 2) ? (q & 1) : (p.strands == 2 ? 1 : 0);
            m = p.lens[r];
            const bool ok = (m >= 1 && m <= p.max_len);
            const uint32_t* rw = p.reads + (int64_t)r * p.stride_words;
            const uint32_t* rn = p.reads_nmask ? p.reads_nmask + (int64_t)r * ((p.stride_words + 1) / 2) : nullptr;
            bool has_n = false;
            if (ok) {
                for (int32_t i = lane; i < m; i += 32) {
                    uint32_t b = read_base(rw, rn, m, i, strand);
                    if (b == 4u && i % istep == 0) has_n = true;        // only scored positions matter
                    sq[q * sq_stride + i] = (uint8_t)b;
                }
            }
            has_n = __any_sync(0xffffffffu, has_n);
            any_n |= has_n;
            const int32_t steps = ok ? (m + istep - 1) / istep : 0;
            // not scanned (bound 0xFFFF): bad lengths, and reads with an N when no tile with the N planes fits
            njq = (ok && !(has_n && ug.b.HALF == 0)) ? (steps + 1) / 2 : 0;
        }
        if (lane == 0) { qnj[q] = njq; qm[q] = m; }
    }
    // ---- the block's tile: the large one, or the one with the N planes if any of its reads holds an N ----------------
    const bool with_n = __syncthreads_or(any_n ? 1 : 0) != 0 && ug.b.HALF != 0;
    const LqTile tg = with_n ? ug.b : ug.a;
    const int32_t NPL = with_n ? LQ_NPL_N : LQ_NPL;
    const int32_t ROWW = tg.ROWW, HALF = tg.HALF, D = 2 * tg.HALF;
    const int32_t CW = HALF / wps;                              // columns of a tile scanned by one warp
    uint32_t* rawp = planes + NPL * ROWW;                       // 2 * NRAW: packed genome words of this tile / the next (cp.async)
    uint32_t* rawn = rawp + 2 * tg.NRAW;                        // 2 * (NRAW / 2 + 1): N-mask words
    const int32_t words_before = NW * 32 + 2 * 32 * LQ_MAX_QSETS + 32 * ug.qsets * TABW + NPL * ROWW + 2 * tg.NRAW + 2 * (tg.NRAW / 2 + 1);
    uint8_t* codes = reinterpret_cast<uint8_t*>(smem + ((words_before + 3) & ~3));   // 16 * NRAW one-hot base codes (16-byte aligned)

    // ---- step 2: this lane's query -> plane offsets in registers -----------------------------------------------------
    // a column is a word (LQ_S16, LQ_F16) or half a word (byte planes: columns 2c, 2c+1 share word c; every offset below is even)
    const int32_t myq = set * 32 + lane;
    const int32_t mynj = qnj[myq], mym = qm[myq];
    const int32_t mystrand = (ns == 2) ? (myq & 1) : (p.strands == 2 ? 1 : 0);
    const uint32_t* myprow = (MODE == LQ_PSSM && myq < nq) ? p.pssm + (int64_t)(r0 + myq / ns) * p.pssm_stride : nullptr;
    uint4* mytab_w = reinterpret_cast<uint4*>(tab) + (size_t)myq * ug.tstride;
    uint2* mytab2 = reinterpret_cast<uint2*>(tab) + (size_t)myq * ug.tstride;
    (void)mystrand; (void)myprow; (void)mytab_w; (void)mytab2;
    // word offset (plane, column) of the operand of double step j for chain 0 of group 0; padding steps: the zero plane
    auto step_word = [&](int32_t j) -> uint32_t {
        uint32_t plane = LQ_ZERO_PLANE, col = 0u;
        if (j < mynj) {
            const int32_t i1 = 2 * j * istep, i2 = i1 + istep;
            const uint32_t b1 = sq[myq * sq_stride + i1];                       // 0..3, 4 = N
            const uint32_t b2 = (i2 < mym) ? sq[myq * sq_stride + i2] : 5u;     // 5 = past the end (pad)
            if (b1 < 4u) plane = b2 < 4u ? b1 * 4u + b2 : (b2 == 5u ? 16u + b1 : 21u + b1);
            else plane = b2 < 4u ? 25u + b2 : (b2 == 5u ? 30u : 29u);
            col = (uint32_t)i1;
        }
        const uint32_t cw = col + ((MODE == LQ_PSSM || TABLE) ? 0u : (uint32_t)(ws * CW));     // column of chain 0, group 0 (tables: of warp 0)
        return plane * (uint32_t)ROWW + (BYTEP ? cw >> 1 : cw);
    };
    uint32_t off[NREG];
    if (TABLE && MODE != LQ_PSSM) {
        // written by the first warp of the query's set, shared by the others (whose column share goes into the group base)
        for (int32_t jp = 0; jp < (ws == 0 ? ug.tstride : 0); jp++)
            mytab2[jp] = make_uint2(step_word(2 * jp) * 4u, step_word(2 * jp + 1) * 4u);
    } else if (MODE != LQ_PSSM) {
#pragma unroll
        for (int j = 0; j < NJ; j++) {
            const uint32_t w = step_word(j);
            if (PACKED) {
                if (j & 1) off[j >> 1] |= w << 16; else off[j >> 1] = w;
            } else {
                off[j] = w * 4u;
            }
        }
    } else {
        // PSSM: the offsets live next to the query's operands in its shared-memory table, one 16-byte entry per double step,
        // written by the first warp of the query's set and shared by the others (whose column share goes into the group base)
        for (int32_t j = 0; j < (ws == 0 ? ug.tstride : 0); j++) {
            uint32_t t01 = 0u, t23 = 0u;
            if (j < mynj) {
                const int32_t i1 = 2 * j, i2 = i1 + 1;
                const uint32_t w1 = pssm_at(myprow, mym, i1, mystrand), w2 = (i2 < mym) ? pssm_at(myprow, mym, i2, mystrand) : 0u;
                const int32_t pm1 = (int16_t)(w1 & 0xFFFFu), px1 = (int16_t)(w1 >> 16), pm2 = (int16_t)(w2 & 0xFFFFu), px2 = (int16_t)(w2 >> 16);
                t01 = ((uint32_t)(px1 + px2) & 0xFFFFu) | ((uint32_t)(pm1 + px2) << 16);      // patterns 0 (neither), 1 (first matches)
                t23 = ((uint32_t)(px1 + pm2) & 0xFFFFu) | ((uint32_t)(pm1 + pm2) << 16);      // 2 (second), 3 (both)
            }
            mytab_w[j] = make_uint4(t01, t23, step_word(j) * 4u, 0u);
        }
    }
    // double steps this warp runs: the longest query of its set, rounded up to the pair the loop body handles
    const int32_t njb = (__reduce_max_sync(0xffffffffu, mynj) + 1) & ~1;

    const uint32_t zero = (uint32_t)p.zero;
    const int32_t tiles_per_frag = (p.F + D - 1) / D;
    const int32_t M = p.match, X = p.mismatch;
    // encodings of the five possible operands: a double step scores 0, 1 or 2 matches, a single step 0 or 1
    const uint32_t e2_0 = lq_enc<MODE>(2 * X), e2_1 = lq_enc<MODE>(M + X), e2_2 = lq_enc<MODE>(2 * M);
    const uint32_t e1_0 = lq_enc<MODE>(X), e1_1 = lq_enc<MODE>(M);
    const char* planes_b = reinterpret_cast<const char*>(planes);
    const uint4* mytab = reinterpret_cast<const uint4*>(tab) + (size_t)myq * ug.tstride;
    (void)mytab;
    uint32_t cur = 0u;                                              // fold threads (tid < 32 * qsets): running fragment maximum
    int32_t prev_f = -1; bool prev_last = false;

    auto fold = [&]() {                                             // previous tile's per-warp maxima -> fragment maximum -> bound
        if (prev_f < 0 || tid >= 32 * ug.qsets) return;
        // thread tid < 32*qsets folds query tid: its set is tid / 32, scanned by warps [set*wps, (set+1)*wps)
        const int32_t fs = tid >> 5;
        uint32_t c = cur;
        for (int32_t w = 0; w < wps; w++) c = max(c, wres[(fs * wps + w) * 32 + lane]);
        if (prev_last) {
            if (tid < nq) {
                const int32_t r = r0 + tid / ns, s = tid % ns;
                uint32_t u = c;                                     // fp16 modes: bit pattern of a non-negative integer value
                if (MODE == LQ_F16 || MODE == LQ_F8) u = (uint32_t)__half2int_rn(__ushort_as_half((unsigned short)c));
                ubound[((int64_t)r * ns + s) * p.n_frag + prev_f] = (qnj[tid] == 0) ? (uint16_t)0xFFFFu : (uint16_t)u;
            }
            c = 0u;
        }
        cur = c;
    };

    // ---- a2, asynchronous half: the raw 2-bit words and N-mask words of a tile travel to shared memory by cp.async
    // (LDGSTS) one tile ahead of the scan; raw word i of a tile is packed word w0 + i, w0 = g0 / 16
    const int32_t n_tiles = (f_end - f_begin) * tiles_per_frag;
    auto prefetch = [&](int32_t it) {
        const int32_t f = f_begin + it / tiles_per_frag, tile = it % tiles_per_frag;
        const int64_t g0 = (int64_t)f * p.F + (int64_t)tile * D;
        const int64_t w0 = g0 >> 4;
        uint32_t* rp = rawp + (it & 1) * tg.NRAW;
        uint32_t* rn = rawn + (it & 1) * (tg.NRAW / 2 + 1);
        for (int32_t i = tid; i < tg.NRAW; i += T) lq_cp_async4(rp + i, p.gpacked + w0 + i);
        for (int32_t i = tid; i < tg.NRAW / 2 + 1; i += T) lq_cp_async4(rn + i, p.gnmask + (w0 >> 1) + i);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if (n_tiles > 0) prefetch(0);

    for (int32_t it = 0; it < n_tiles; it++) {
        const int32_t f = f_begin + it / tiles_per_frag, tile = it % tiles_per_frag;
        const int64_t fstart = (int64_t)f * p.F;
        const int64_t trunc = (p.V < 0) ? (int64_t)0x7FFFFFFFFFFFFFFFll : fstart + p.F + p.V;
        {
            const int32_t toff = tile * D;
            const int64_t g0 = fstart + toff;
            const int32_t nvalid = min(D, p.F - toff);
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncthreads();                                        // previous tile scanned (planes free, wres complete); raw words landed
            fold();
            // ---- a2: raw words -> one byte per genome position: one-hot of the base (1, 2, 4, 8), 0 = N or not readable
            {
                const uint32_t* rp = rawp + (it & 1) * tg.NRAW;
                const uint32_t* rn = rawn + (it & 1) * (tg.NRAW / 2 + 1);
                const int64_t w0 = g0 >> 4;
                for (int32_t i = tid; i < tg.NRAW; i += T) {
                    const uint32_t w = rp[i];
                    const int64_t W = w0 + i;
                    const uint32_t mk = (rn[(int32_t)((W >> 1) - (w0 >> 1))] >> (16u * (uint32_t)(W & 1))) & 0xFFFFu;
                    const int64_t pos0 = W << 4;
                    uint32_t out[4];
#pragma unroll
                    for (int b = 0; b < 16; b++) {
                        const uint32_t c = (w >> (2 * b)) & 3u;
                        const bool dead = ((mk >> b) & 1u) || (pos0 + b >= trunc);
                        const uint32_t oh = dead ? 0u : (1u << c);
                        if ((b & 3) == 0) out[b >> 2] = oh; else out[b >> 2] |= oh << (8 * (b & 3));
                    }
                    *reinterpret_cast<uint4*>(codes + 16 * i) = make_uint4(out[0], out[1], out[2], out[3]);
                }
            }
            if (it + 1 < n_tiles) prefetch(it + 1);
            __syncthreads();
            // ---- a2: codes -> dibase planes ----------------------------------------------------------------------
            const int32_t sh = (int32_t)(g0 & 15);                  // codes[sh + x] = genome position g0 + x
            if (!BYTEP) {
                for (int32_t x = tid; x < tg.COLS; x += T) {
                    const uint32_t lo1 = codes[sh + x], lo2 = codes[sh + x + istep];
                    const uint32_t hi1 = codes[sh + x + HALF], hi2 = codes[sh + x + HALF + istep];
#pragma unroll
                    for (uint32_t c1 = 0; c1 < 4; c1++) {
                        const uint32_t ml = (lo1 >> c1) & 1u, mh = (hi1 >> c1) & 1u;
#pragma unroll
                        for (uint32_t c2 = 0; c2 < 4; c2++) {
                            const uint32_t nl = ml + ((lo2 >> c2) & 1u), nh = mh + ((hi2 >> c2) & 1u);
                            const uint32_t vl = nl == 2 ? e2_2 : (nl == 1 ? e2_1 : e2_0), vh = nh == 2 ? e2_2 : (nh == 1 ? e2_1 : e2_0);
                            planes[(c1 * 4 + c2) * ROWW + x] = vl | (vh << 16);
                        }
                        planes[(16 + c1) * ROWW + x] = (ml ? e1_1 : e1_0) | ((mh ? e1_1 : e1_0) << 16);
                        if (with_n) {                               // (c1, N): the second position never matches; (N, c): the first
                            planes[(21 + c1) * ROWW + x] = (ml ? e2_1 : e2_0) | ((mh ? e2_1 : e2_0) << 16);
                            planes[(25 + c1) * ROWW + x] = (((lo2 >> c1) & 1u) ? e2_1 : e2_0) | ((((hi2 >> c1) & 1u) ? e2_1 : e2_0) << 16);
                        }
                    }
                    planes[LQ_ZERO_PLANE * ROWW + x] = 0u;
                    if (with_n) { planes[29 * ROWW + x] = e2_0 | (e2_0 << 16); planes[30 * ROWW + x] = e1_0 | (e1_0 << 16); }
                }
            } else {
                // word xw = columns 2xw, 2xw + 1, bytes (lo, hi, lo', hi').  The four lanes' one-hot codes go into the four
                // nibbles of a 16-bit value; (OH >> c) & 0x1111 is then the lanes' match flag against base c, the sum of two
                // such values their match count (0..2 per nibble), and one PRMT with that value as the selector maps every
                // count to its operand byte: 3 instructions per plane word
                // PSSM: the byte is the PRMT selector of the match pattern p = first + 2 * second, (2p + 1) << 4 | 2p
                const uint32_t tab2 = MODE == LQ_PSSM ? 0x76543210u : (e2_0 >> 8) | (e2_1 & 0xFF00u) | ((e2_2 & 0xFF00u) << 8);
                const uint32_t tab1 = MODE == LQ_PSSM ? 0x76543210u : (e1_0 >> 8) | (e1_1 & 0xFF00u);
                const uint32_t second = MODE == LQ_PSSM ? 2u : 1u;  // weight of the second position in the table index
                for (int32_t xw = tid; xw < tg.COLS / 2; xw += T) {
                    const uint8_t* c0 = codes + sh + 2 * xw;
                    const uint32_t oh1 = c0[0] | (c0[HALF] << 4) | (c0[1] << 8) | (c0[HALF + 1] << 12);
                    const uint32_t oh2 = c0[istep] | (c0[HALF + istep] << 4) | (c0[1 + istep] << 8) | (c0[HALF + 1 + istep] << 12);
                    uint32_t A[4], Bm[4];
#pragma unroll
                    for (int c = 0; c < 4; c++) { A[c] = (oh1 >> c) & 0x1111u; Bm[c] = (oh2 >> c) & 0x1111u; }
#pragma unroll
                    for (uint32_t c1 = 0; c1 < 4; c1++) {
#pragma unroll
                        for (uint32_t c2 = 0; c2 < 4; c2++)
                            planes[(c1 * 4 + c2) * ROWW + xw] = lq_prmt(tab2, 0u, A[c1] + second * Bm[c2]);
                        planes[(16 + c1) * ROWW + xw] = lq_prmt(tab1, 0u, A[c1]);
                        if (with_n) {                               // (c1, N): the second position never matches; (N, c): the first
                            planes[(21 + c1) * ROWW + xw] = lq_prmt(tab2, 0u, A[c1]);
                            planes[(25 + c1) * ROWW + xw] = lq_prmt(tab2, 0u, second * Bm[c1]);
                        }
                    }
                    planes[LQ_ZERO_PLANE * ROWW + xw] = MODE == LQ_PSSM ? 0x10101010u : 0u;      // PSSM: pattern 0 of an all-zero table
                    if (with_n) {
                        planes[29 * ROWW + xw] = MODE == LQ_PSSM ? 0x10101010u : (e2_0 >> 8) * 0x01010101u;
                        planes[30 * ROWW + xw] = MODE == LQ_PSSM ? 0x10101010u : (e1_0 >> 8) * 0x01010101u;
                    }
                }
            }
            __syncthreads();

            // ---- a3: this lane's query against the warp's columns of the tile --------------------------------------
            uint32_t tmax = 0u;
            for (int32_t g = 0; g < tg.NG; g++) {
                const char* pg = planes_b + g * (BYTEP ? K * 2 : K * 4)
                               + ((MODE == LQ_PSSM || TABLE) ? ws * CW * (BYTEP ? 2 : 4) : 0);   // warp-uniform group base
                uint32_t H[K], B[K];
#pragma unroll
                for (int k = 0; k < K; k++) { H[k] = 0u; B[k] = 0u; }
                // two double steps of the K chains: operands at byte offsets o0, o1 of the group's columns (PSSM: tq = the
                // query's four operands of either double step)
                auto pair = [&](uint32_t o0, uint32_t o1, const uint4& tq) {
                    uint32_t Ha[K], v[K];
                    if (MODE == LQ_PSSM) {
#pragma unroll
                        for (int k = 0; k < K; k += 2) {
                            const uint32_t w = *reinterpret_cast<const uint32_t*>(pg + o0 + k * 2);
                            v[k] = lq_prmt(tq.x, tq.y, w); v[k + 1] = lq_prmt(tq.x, tq.y, lq_hi16(w));
                        }
                    } else if (MODE == LQ_F8) {
#pragma unroll
                        for (int k = 0; k < K; k += 2) {
                            const uint32_t w = *reinterpret_cast<const uint32_t*>(pg + o0 + k * 2);
                            v[k] = __byte_perm(w, 0u, 0x1404); v[k + 1] = __byte_perm(w, 0u, 0x3424);
                        }
                    } else {
#pragma unroll
                        for (int k = 0; k < K; k++) v[k] = *reinterpret_cast<const uint32_t*>(pg + o0 + k * 4);
                    }
#pragma unroll
                    for (int k = 0; k < K; k++) {
                        if (MODE == LQ_S16 || MODE == LQ_PSSM) Ha[k] = __viaddmax_s16x2(H[k], v[k], zero);
                        else asm("fma.rn.relu.f16x2 %0, %1, %2, %3;" : "=r"(Ha[k]) : "r"(H[k]), "r"(0x3C003C00u), "r"(v[k]));
                    }
                    if (MODE == LQ_PSSM) {
#pragma unroll
                        for (int k = 0; k < K; k += 2) {
                            const uint32_t w = *reinterpret_cast<const uint32_t*>(pg + o1 + k * 2);
                            v[k] = lq_prmt(tq.z, tq.w, w); v[k + 1] = lq_prmt(tq.z, tq.w, lq_hi16(w));
                        }
                    } else if (MODE == LQ_F8) {
#pragma unroll
                        for (int k = 0; k < K; k += 2) {
                            const uint32_t w = *reinterpret_cast<const uint32_t*>(pg + o1 + k * 2);
                            v[k] = __byte_perm(w, 0u, 0x1404); v[k + 1] = __byte_perm(w, 0u, 0x3424);
                        }
                    } else {
#pragma unroll
                        for (int k = 0; k < K; k++) v[k] = *reinterpret_cast<const uint32_t*>(pg + o1 + k * 4);
                    }
#pragma unroll
                    for (int k = 0; k < K; k++) {
                        if (MODE == LQ_S16 || MODE == LQ_PSSM) H[k] = __viaddmax_s16x2(Ha[k], v[k], zero);
                        else asm("fma.rn.relu.f16x2 %0, %1, %2, %3;" : "=r"(H[k]) : "r"(Ha[k]), "r"(0x3C003C00u), "r"(v[k]));
                    }
#pragma unroll
                    for (int k = 0; k < K; k++) B[k] = __vimax3_s16x2(B[k], Ha[k], H[k]);
                };
                if (MODE == LQ_PSSM) {
                    // the query's table entry of a double step = (operands 0/1, operands 2/3, plane offset, -): one LDS.128
#pragma unroll 2
                    for (int32_t j = 0; j < njb; j += 2) {
                        const uint4 ta = mytab[j], tb = mytab[j + 1];
                        pair(ta.z, tb.z, make_uint4(ta.x, ta.y, tb.x, tb.y));
                    }
                } else if (TABLE) {
#pragma unroll 4
                    for (int32_t jp = 0; jp < (njb >> 1); jp++) {
                        const uint2 o = mytab2[jp];
                        pair(o.x, o.y, make_uint4(0u, 0u, 0u, 0u));
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < NJ; j += 2) {
                        if ((j & 7) == 0 && j >= njb) break;        // padding steps add 0: the check only saves time, so it is coarse
                        uint32_t o0, o1;
                        if (PACKED) {                               // volatile: unpacked per use, or the compiler hoists all NJ results out of the group loop and spills them
                            uint32_t lo, hi;
                            asm volatile("and.b32 %0, %1, 0xFFFF;" : "=r"(lo) : "r"(off[j >> 1]));
                            asm volatile("shr.u32 %0, %1, 16;" : "=r"(hi) : "r"(off[j >> 1]));
                            o0 = lo << 2; o1 = hi << 2;
                        }
                        else { o0 = off[j]; o1 = off[j + 1]; }
                        pair(o0, o1, make_uint4(0u, 0u, 0u, 0u));
                    }
                }
                if (nvalid < D) {                                   // ragged last tile of a fragment: drop foreign window starts
                    const int32_t x0 = ws * CW + g * K;
#pragma unroll
                    for (int k = 0; k < K; k++) {
                        if (x0 + k >= nvalid) B[k] &= 0xFFFF0000u;
                        if (x0 + k + HALF >= nvalid) B[k] &= 0x0000FFFFu;
                    }
                }
#pragma unroll
                for (int k = 0; k < K; k += 2) tmax = __vimax3_s16x2(tmax, B[k], B[k + 1]);
            }
            wres[warp * 32 + lane] = max(tmax & 0xFFFFu, tmax >> 16);
            prev_f = f; prev_last = (tile == tiles_per_frag - 1);
        }
    }
    __syncthreads();
    fold();
}

// every value a plane can hold, as an e5m2 byte (= the high byte of its fp16 form), must be exact
bool lq_e5m2_exact(int32_t v)
{
    if (v < 0) v = -v;
    if (v == 0) return true;
    if (v > 57344) return false;                                // the largest finite e5m2 value
    while ((v & 1) == 0) v >>= 1;
    return v < 8;                                               // three significant bits (1.xx)
}

struct LqSmem { int32_t ROWW, COLS, NRAW; size_t bytes; };
// PSSM: table entries per thread: the double steps of the longest read, rounded up to the pair the loop handles, made odd
int32_t lq_tstride(int32_t max_len, int32_t istep)
{
    int32_t steps = (max_len + istep - 1) / istep;
    return ((((steps + 1) / 2) + 1) & ~1) | 1;
}
// TABLE: entries (pairs of double steps) per query, made odd
int32_t lq_pstride(int32_t max_len, int32_t istep)
{
    int32_t steps = (max_len + istep - 1) / istep;
    return ((((steps + 1) / 2) + 1) / 2) | 1;
}
LqSmem lq_smem(int32_t half, int32_t max_len, int32_t istep, int modef, int npl, int32_t qsets)
{
    const int mode = modef & 7;
    // columns read: chain column < HALF, plus the column of the last double step (< max_len rounded up to even steps)
    LqSmem s;
    int32_t halo = ((max_len + 2 * istep + 3) & ~3);
    s.COLS = half + halo;
    int32_t roww = (mode == LQ_F8 || mode == LQ_PSSM) ? s.COLS / 2 : s.COLS;
    roww += (33 - (roww & 31)) & 31;                            // 1 (mod 32): plane p, word c -> bank (p + c) mod 32
    s.ROWW = roww;
    // genome positions a tile reads: [g0, g0 + HALF + COLS + istep), from the 16-aligned position below g0
    s.NRAW = ((half + s.COLS + istep + 15 + 15) / 16 + 1) & ~1;
    // planes, wres, qnj + qm, raw words (2 buffers), raw mask words (2 buffers), pad to 16 bytes, codes
    size_t words = (size_t)npl * roww + LQ_NW * 32 + 2 * 32 * LQ_MAX_QSETS + 2 * s.NRAW + 2 * (s.NRAW / 2 + 1);
    if (mode == LQ_PSSM) words += (size_t)32 * qsets * 4 * lq_tstride(max_len, istep);     // per-query (operands, offset) tables
    else if (modef & LQ_TABLE) words += (size_t)32 * qsets * 2 * lq_pstride(max_len, istep);   // per-query offset-pair tables
    words = (words + 3) & ~(size_t)3;
    s.bytes = words * 4 + (size_t)16 * s.NRAW;
    return s;
}

thread_local int t_lq_qsets = 0;       // tuning hook: query sets per block (reads per block = 16 * qsets with both strands); 0 = by batch size
thread_local int t_lq_half = 0;        // tuning hook: force the tile (0 = automatic)
thread_local int t_lq_mode = -1;       // tuning hook: force the arithmetic (-1 = automatic)
thread_local bool t_lq_k8 = false;     // tuning hook: 8 chains per thread even for short reads
thread_local int t_lq_table = -1;      // tuning hook: plane offsets from the shared-memory table (1), in registers (0), automatic (-1)

int lq_mode(const ScanParams& p)
{
    if (p.pssm) return LQ_PSSM;
    const int32_t M = p.match, X = p.mismatch;
    const bool f16_ok = (int64_t)p.max_len * M <= 2048 && 2 * M <= 2048 && -2 * X <= 2048;
    const bool f8_ok = f16_ok && lq_e5m2_exact(2 * M) && lq_e5m2_exact(M + X) && lq_e5m2_exact(2 * X) && lq_e5m2_exact(M) &&
                       lq_e5m2_exact(X);
    int want = t_lq_mode >= 0 ? t_lq_mode : LQ_F8;
    if (want == LQ_F8 && !f8_ok) want = LQ_F16;
    if (want == LQ_F16 && !f16_ok) want = LQ_S16;
    return want;
}

int32_t lq_double_steps(const ScanParams& p);
int32_t lq_nj_instance(int32_t nj, int mode);

// arithmetic | LQ_TABLE: where a query's plane offsets live.  Registers hold at most 128 double steps (256 scored positions);
// beyond that, and where it measured faster, they come from the shared-memory table.  Measured (e5m2 operands, cells/clk/SM,
// registers / table): 36 bp 129.8 / 118.2, 100 bp 136.7 / 124.5, 150 bp 133.1 / 125.3, 250 bp 112.1 (16-bit offset pairs) /
// 126.5: the table costs one LDS.64 per pair of double steps and a rolled loop, and is the same for every length.  With 16 chains
// per thread (the table frees the registers for them) it reaches 131.5 / 131.6 / 132.8 at 100 / 150 / 250 bp.
int lq_plan(const ScanParams& p)
{
    const int mode = lq_mode(p);
    if (mode == LQ_PSSM) return mode | (t_lq_k8 ? 0 : LQ_K16);   // table-driven by construction: registers for 16 chains
    const int32_t nj = lq_double_steps(p);
    bool table = nj > LQ_TABLE_FROM_NJ;
    if (t_lq_table == 1) table = true;
    if (t_lq_table == 0 && nj <= 128) table = false;
    if (nj > 128) table = true;
    const int32_t inst = lq_nj_instance(nj, mode);              // only the tight short-read instances exist with 16 chains
    const bool k16 = !table && mode == LQ_F8 && nj <= LQ_K16_UP_TO_NJ && (inst == 18 || inst == 26 || inst == 38) && !t_lq_k8;
    const bool t16 = table && mode == LQ_F8 && !t_lq_k8;         // the table-driven e5m2 instance has the registers for 16 chains too
    return mode | (table ? LQ_TABLE : 0) | ((k16 || t16) ? LQ_K16 : 0);
}

// the tile: 2*HALF window starts, HALF a multiple of the columns one more group of every warp of a set adds;
// least padding of the fragment length first, larger tiles on ties; two blocks per SM must fit
bool lq_pick_tile(const mss_genome* g, const ScanParams& p, int32_t qsets, int mode, int npl, int32_t forced_half, LqTile* out, size_t* bytes)
{
    const int32_t unit = (LQ_NW / qsets) * ((mode & LQ_K16) ? 16 : LQ_K);
    const size_t prologue = (size_t)32 * qsets * ((p.max_len + 3) & ~3);
    int32_t best = 0; double best_waste = 1e30;
    for (int32_t half = unit; half <= 4096; half += unit) {
        if (forced_half > 0 && half != forced_half) continue;
        if (half < 128) continue;
        LqSmem s = lq_smem(half, p.max_len, p.istep, mode, npl, qsets);
        if (s.bytes * LQ_BLOCKS_PER_SM + 2048 * LQ_BLOCKS_PER_SM > (size_t)g->max_smem_optin) break;
        if ((size_t)npl * s.ROWW * 4 < prologue) continue;         // the prologue borrows the plane area
        if ((int64_t)npl * s.ROWW + 4096 > 65535) break;             // packed 16-bit word offsets
        int32_t D = 2 * half;
        double waste = (double)((g->frag_len + D - 1) / D) * D / g->frag_len;
        waste *= 1.0 + 0.02 * (double)(s.COLS - half) / half;       // look-ahead columns are staged, not scanned: mild preference for large tiles
        if (waste < best_waste - 1e-9) { best_waste = waste; best = half; }
    }
    if (!best) return false;
    LqSmem s = lq_smem(best, p.max_len, p.istep, mode, npl, qsets);
    if (out) { out->HALF = best; out->ROWW = s.ROWW; out->COLS = s.COLS; out->NRAW = s.NRAW; out->NG = best / unit; }
    if (bytes) *bytes = s.bytes;
    return true;
}

// both tiles of a launch: the one of N-free blocks decides whether the kernel applies at all
bool lq_pick(const mss_genome* g, const ScanParams& p, int32_t qsets, int mode, LqGeom* out, size_t* bytes)
{
    LqTile a, b;
    size_t ba = 0, bb = 0;
    if (!lq_pick_tile(g, p, qsets, mode, LQ_NPL, t_lq_half, &a, &ba)) return false;
    if (!lq_pick_tile(g, p, qsets, mode, LQ_NPL_N, 0, &b, &bb)) { b = LqTile{0, 0, 0, 0, 0}; bb = 0; }
    if (out) { out->a = a; out->b = b; out->qsets = qsets; out->tstride = (mode & LQ_TABLE) ? lq_pstride(p.max_len, p.istep) : lq_tstride(p.max_len, p.istep); }
    if (bytes) *bytes = ba > bb ? ba : bb;
    return true;
}

// query sets per block: more sets amortise the tile staging over more queries (measured, cells/clk/SM with 1 / 2 / 4 sets:
// 133.4 / 135.5 / 136.8 at 100 bp, 121.5 / 126.6 / 129.8 at 36 bp, 122.2 / 123.6 / 124.5 at 150 bp): the most sets with which
// the grid (read groups x fragments) still fills the GPU's ~48 waves of resident blocks
int32_t lq_qsets(const mss_genome* g, const ScanParams& p)
{
    if (p.pssm) return 1;                                       // the per-query tables take the room more query sets would need
    if (t_lq_qsets) return t_lq_qsets;
    int32_t most = 4;                                           // offset tables: at most 40 kB of them beside the tile
    if (lq_plan(p) & LQ_TABLE)
        while (most > 1 && (size_t)32 * most * 8 * lq_pstride(p.max_len, p.istep) > 40960) most >>= 1;
    const int64_t queries = (int64_t)p.n_reads * (p.strands == 3 ? 2 : 1);
    const int64_t target = (int64_t)g->sm_count * LQ_BLOCKS_PER_SM * 48;
    for (int32_t qs = most; qs > 1; qs >>= 1)
        if (((queries + 32 * qs - 1) / (32 * qs)) * (int64_t)g->n_frag >= target) return qs;
    return 1;
}

// the kernel instance (most double steps held) that serves queries of up to nj double steps
int32_t lq_nj_instance(int32_t nj, int mode)
{
    if (mode == LQ_F8) {
        if (nj <= 18) return 18;
        if (nj <= 26) return 26;
        if (nj > 32 && nj <= 38) return 38;
    }
    if (mode == LQ_F8 && nj > 38 && nj <= 50) return 50;
    if (mode == LQ_F8 && nj > 64 && nj <= 76) return 76;
    if (nj <= 32) return 32;
    if (nj <= 64) return 64;
    if (nj <= 80) return 80;
    return 128;
}

int32_t lq_double_steps(const ScanParams& p)
{
    int32_t steps = (p.max_len + p.istep - 1) / p.istep;
    return (steps + 1) / 2;
}

template <int NJ, bool PACKED, int MODE, int KC = LQ_K>
cudaError_t lq_launch3(const ScanParams& p, const LqGeom& ug, uint16_t* ubound, cudaStream_t st, size_t smem)
{
    cudaError_t e = cudaFuncSetAttribute(scan_filter_lq_kernel<NJ, PACKED, MODE, KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int64_t blocks = (int64_t)ug.n_groups * ug.n_splits;
    scan_filter_lq_kernel<NJ, PACKED, MODE, KC><<<(unsigned)blocks, 32 * LQ_NW, smem, st>>>(p, ug, ubound);
    return cudaGetLastError();
}

template <int NJ, bool PACKED>
cudaError_t lq_launch(int mode, const ScanParams& p, const LqGeom& ug, uint16_t* ubound, cudaStream_t st, size_t smem)
{
    if (mode == LQ_F8) return lq_launch3<NJ, PACKED, LQ_F8>(p, ug, ubound, st, smem);
    if (mode == LQ_F16) return lq_launch3<NJ, PACKED, LQ_F16>(p, ug, ubound, st, smem);
    return lq_launch3<NJ, PACKED, LQ_S16>(p, ug, ubound, st, smem);
}

}  // namespace

void scan_filter_lq_tune(int qsets, int half, int mode)
{
    t_lq_qsets = (qsets == 1 || qsets == 2 || qsets == 4) ? qsets : 0;
    t_lq_half = half > 0 ? half : 0;
    // mode: -1 automatic; 0..2 the arithmetic; + 8 = offsets from the table, + 16 = offsets in registers (3 = automatic arithmetic)
    t_lq_table = -1; t_lq_k8 = false;
    if (mode >= 32) { t_lq_k8 = true; mode -= 32; if (mode == 3) mode = -1; }
    if (mode >= 16) { t_lq_table = 0; mode -= 16; } else if (mode >= 8) { t_lq_table = 1; mode -= 8; }
    t_lq_mode = (mode >= 0 && mode <= 2) ? mode : -1;
}

bool scan_filter_lq_supported(const mss_genome* g, const ScanParams& p)
{
    if (p.pssm && p.istep != 1) return false;
    return lq_pick(g, p, lq_qsets(g, p), lq_plan(p), nullptr, nullptr);      // no tile fits (very long reads): the tile kernel of scan_filter.cu
}

cudaError_t launch_scan_filter_lq(const mss_genome* g, const ScanParams& p, uint16_t* ubound, cudaStream_t st, int32_t* grid_out,
                                  int32_t* smem_out, int32_t* tile_out, int32_t* rpb_out, int32_t* kind_out)
{
    LqGeom ug;
    const int plan = lq_plan(p), mode = plan & 7;
    if (kind_out) *kind_out = ((plan & LQ_TABLE) ? 6 : 2) + mode;
    size_t smem = 0;
    if (!lq_pick(g, p, lq_qsets(g, p), plan, &ug, &smem)) return cudaErrorInvalidConfiguration;
    const int32_t ns = p.strands == 3 ? 2 : 1;
    ug.reads_per_group = 32 * ug.qsets / ns;
    ug.n_groups = (p.n_reads + ug.reads_per_group - 1) / ug.reads_per_group;
    if (ug.n_groups < 1) ug.n_groups = 1;
    int64_t target = (int64_t)g->sm_count * 2 * 48;             // ~48 waves of the 2 resident blocks per SM
    int64_t want = (target + ug.n_groups - 1) / ug.n_groups;
    if (want < 1) want = 1;
    if (want > g->n_frag) want = g->n_frag;
    ug.frags_per_split = (int32_t)((g->n_frag + want - 1) / want);
    ug.n_splits = (g->n_frag + ug.frags_per_split - 1) / ug.frags_per_split;
    if (grid_out) *grid_out = (int32_t)((int64_t)ug.n_groups * ug.n_splits);
    if (smem_out) *smem_out = (int32_t)smem;
    if (tile_out) *tile_out = 2 * ug.a.HALF;
    if (rpb_out) *rpb_out = ug.reads_per_group;
    // padding steps cost time (the early-exit check is coarse): the common read lengths get a tight instance of the
    // fast arithmetic (36, 51, 76, 100, 150 bp)
    if (mode == LQ_PSSM)                                                                  // table-driven: one instance for every length
        return (plan & LQ_K16) ? lq_launch3<2, false, LQ_PSSM, 16>(p, ug, ubound, st, smem) : lq_launch3<2, false, LQ_PSSM>(p, ug, ubound, st, smem);
    if ((plan & LQ_TABLE) && (plan & LQ_K16)) return lq_launch3<0, false, LQ_F8, 16>(p, ug, ubound, st, smem);
    if (plan & LQ_TABLE) return lq_launch<0, false>(mode, p, ug, ubound, st, smem);
    switch (lq_nj_instance(lq_double_steps(p), mode)) {
        case 18: return (plan & LQ_K16) ? lq_launch3<18, false, LQ_F8, 16>(p, ug, ubound, st, smem) : lq_launch3<18, false, LQ_F8>(p, ug, ubound, st, smem);
        case 26: return (plan & LQ_K16) ? lq_launch3<26, false, LQ_F8, 16>(p, ug, ubound, st, smem) : lq_launch3<26, false, LQ_F8>(p, ug, ubound, st, smem);
        case 38: return (plan & LQ_K16) ? lq_launch3<38, false, LQ_F8, 16>(p, ug, ubound, st, smem) : lq_launch3<38, false, LQ_F8>(p, ug, ubound, st, smem);
        case 50: return lq_launch3<50, false, LQ_F8>(p, ug, ubound, st, smem);     // 16 chains measured slower here (135.3 against 136.7)
        case 76: return lq_launch3<76, false, LQ_F8>(p, ug, ubound, st, smem);
        case 32: return lq_launch<32, false>(mode, p, ug, ubound, st, smem);
        case 64: return lq_launch<64, false>(mode, p, ug, ubound, st, smem);
        case 80: return lq_launch<80, false>(mode, p, ug, ubound, st, smem);
        default: break;
    }
    return lq_launch<128, true>(mode, p, ug, ubound, st, smem);
}
