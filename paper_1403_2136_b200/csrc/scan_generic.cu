// Generic MaxSS scan: correct for every (F, V, m); one block per (read, fragment), int32 scores, no tiling.
// It is the fallback for geometries the DPX tile kernel does not take (F < 512) and the in-library cross-check
// variant (mss_set_scan_variant(1)).  PAPER.md:41 (Kadane), :57 (thread <-> fragment sliding window, top-2).
#include "mss_common.cuh"

#define GEN_THREADS 128

__global__ void __launch_bounds__(GEN_THREADS)
scan_generic_kernel(ScanParams p, int32_t read0, int32_t chunk_reads, uint64_t* __restrict__ fragkey)
{
    extern __shared__ __align__(8) uint8_t gsm[];
    int32_t* qs = reinterpret_cast<int32_t*>(gsm);      // PSSM only: (pmatch, pmismatch) of the strand-oriented read
    uint8_t* q = gsm + (p.pssm ? (size_t)p.max_len * 8 : 0);   // strand-oriented read, one byte per base
    __shared__ uint64_t wmax[GEN_THREADS / 32];
    int64_t bid = blockIdx.x;
    int32_t rl = (int32_t)(bid % chunk_reads);
    int32_t f = (int32_t)(bid / chunk_reads);
    int32_t r = read0 + rl;
    int32_t m = p.lens[r];
    uint64_t best = 0;                                   // key of (score 0, reverse, diag max) is never below a real one
    bool any = false;
    if (m >= 1 && m <= p.max_len) {
        const uint32_t* rw = p.reads + (int64_t)r * p.stride_words;
        const uint32_t* rn = p.reads_nmask ? p.reads_nmask + (int64_t)r * ((p.stride_words + 1) / 2) : nullptr;
        const uint32_t* prow = p.pssm ? p.pssm + (int64_t)r * p.pssm_stride : nullptr;
        int32_t veff = (p.V < 0 || p.V > m - 1) ? m - 1 : p.V;
        int64_t fstart = (int64_t)f * p.F, end = fstart + p.F + veff;
        for (int32_t s = 0; s < 2; s++) {
            if (!(p.strands & (1 << s))) continue;
            __syncthreads();
            for (int32_t i = threadIdx.x; i < m; i += GEN_THREADS) {
                q[i] = (uint8_t)read_base(rw, rn, m, i, s);
                if (prow) {
                    uint32_t w = pssm_at(prow, m, i, s);
                    qs[2 * i] = (int32_t)(int16_t)(w & 0xFFFFu);
                    qs[2 * i + 1] = (int32_t)(int16_t)(w >> 16);
                }
            }
            __syncthreads();
            for (int32_t d = threadIdx.x; d < p.F; d += GEN_THREADS) {
                int64_t g = fstart + d;
                int32_t n = (end - g < m) ? (int32_t)(end - g) : m;
                int32_t H = 0, b = 0;
                for (int32_t i = 0; i < n; i += p.istep) {
                    uint32_t gb = base_at(p.gpacked, p.gnmask, g + i);
                    bool eq = gb < 4u && gb == q[i];
                    int32_t sc = prow ? (eq ? qs[2 * i] : qs[2 * i + 1]) : (eq ? p.match : p.mismatch);
                    H = max(H + sc, 0);
                    b = max(b, H);
                }
                uint64_t k = frag_key(b, s, d);
                if (!any || k > best) { best = k; any = true; }
            }
        }
    }
    // block max (threads without a diagonal carry key 0, below every real key since diag <= 0x7FFFFFFF-... > 0)
    uint64_t k = any ? best : 0ull;
    for (int off = 16; off; off >>= 1) {
        uint64_t o = __shfl_xor_sync(0xffffffffu, k, off);
        k = o > k ? o : k;
    }
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = k;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < GEN_THREADS / 32; w++) k = wmax[w] > k ? wmax[w] : k;
        fragkey[(int64_t)f * chunk_reads + rl] = k;
    }
}

__global__ void top2_over_fragments_kernel(ScanParams p, int32_t read0, int32_t chunk_reads,
                                           const uint64_t* __restrict__ fragkey, mss_top2_t* __restrict__ out)
{
    int32_t rl = blockIdx.x * blockDim.x + threadIdx.x;
    if (rl >= chunk_reads) return;
    int32_t r = read0 + rl;
    mss_hit_t none = { -1, 0, 0, 0 };
    mss_hit_t best = none, second = none;
    int32_t m = p.lens[r];
    if (m >= 1 && m <= p.max_len) {
        for (int32_t f = 0; f < p.n_frag; f++) {
            uint64_t k = fragkey[(int64_t)f * chunk_reads + rl];
            mss_hit_t h; h.frag = f;
            frag_key_unpack(k, h.score, h.strand, h.diag);
            top2_push(best, second, h);
        }
    }
    out[r].best = best;
    out[r].second = second;
}

static int32_t generic_chunk(const mss_genome* g, int32_t n_reads)
{
    int64_t per_read = (int64_t)g->n_frag * 8;
    int64_t c = (256ll << 20) / per_read;
    if (c < 1) c = 1;
    if (c > n_reads) c = n_reads;
    // grid.x limit 2^31-1
    int64_t maxc = 2147483647ll / g->n_frag;
    if (c > maxc) c = maxc;
    if (c < 1) c = 1;
    return (int32_t)c;
}

size_t scan_generic_workspace(const mss_genome* g, int32_t n_reads)
{
    if (n_reads <= 0) return 256;
    return (size_t)generic_chunk(g, n_reads) * (size_t)g->n_frag * 8 + 256;
}

cudaError_t launch_scan_generic(const mss_genome* g, const ScanParams& p, void* ws, size_t ws_bytes,
                                mss_top2_t* d_out, cudaStream_t st, mss_launch_info_t* info)
{
    int32_t chunk = generic_chunk(g, p.n_reads);
    uint64_t* fragkey = (uint64_t*)ws;
    int launches = 0;
    {
        size_t smem = (size_t)p.max_len + 16 + (p.pssm ? (size_t)p.max_len * 8 : 0);
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(scan_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
    }
    for (int32_t r0 = 0; r0 < p.n_reads; r0 += chunk) {
        int32_t c = p.n_reads - r0 < chunk ? p.n_reads - r0 : chunk;
        int64_t blocks = (int64_t)c * g->n_frag;
        size_t smem = (size_t)p.max_len + 16 + (p.pssm ? (size_t)p.max_len * 8 : 0);
        scan_generic_kernel<<<(unsigned)blocks, GEN_THREADS, smem, st>>>(p, r0, c, fragkey);
        top2_over_fragments_kernel<<<(c + 127) / 128, 128, 0, st>>>(p, r0, c, fragkey, d_out);
        launches += 2;
        if (info) { info->grid = (int32_t)blocks; }
    }
    if (info) {
        info->variant = 1; info->block = GEN_THREADS; info->smem_bytes = p.max_len + 16;
        info->reads_per_block = 1; info->tile_diagonals = g->frag_len; info->launches = launches; info->pass1_kernel = 0;
    }
    return cudaGetLastError();
}
