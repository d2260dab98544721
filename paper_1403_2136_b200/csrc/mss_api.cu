// C ABI of include/mss.h: argument checks, handle, variant dispatch.  No compute lives here.
#include <cmath>
#include <new>
#include "mss_common.cuh"

namespace {
thread_local int t_last_cuda = 0;
thread_local int t_variant = 0;
thread_local mss_launch_info_t t_info = { 0, 0, 0, 0, 0, 0, 0, 0 };

int cuda_fail(cudaError_t e) { t_last_cuda = (int)e; return MSS_ERR_CUDA; }

int64_t padded_len(int64_t n_bases, int32_t frag_len)
{
    int64_t nfrag = (n_bases + frag_len - 1) / frag_len;
    int64_t need = nfrag * frag_len + 8192 + MSS_MAX_READ_LEN + 128;
    return (need + 127) / 128 * 128;
}

// the handle belongs to the device that was current at mss_genome_load: its pointers, SM count and shared-memory limit
// mean nothing elsewhere, so a call made with another device current is refused instead of launched
int check_device(const mss_genome* g)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    return dev == g->device ? MSS_OK : MSS_ERR_ARG;
}

int check_scoring_scan(mss_scoring_t sc, int32_t max_len)
{
    if (sc.match <= 0 || sc.mismatch >= 0) return MSS_ERR_RANGE;
    if (max_len > MSS_MAX_READ_LEN) return MSS_ERR_RANGE;
    if ((int64_t)max_len * sc.match > 32767 || sc.mismatch < -32768) return MSS_ERR_RANGE;
    return MSS_OK;
}
}  // namespace

int mss_record_cuda_error(cudaError_t e) { return cuda_fail(e); }

extern "C" {

size_t mss_genome_workspace_bytes(int64_t n_bases, int32_t frag_len, int32_t overlap)
{
    if (n_bases <= 0 || frag_len <= 0 || overlap < -1) return 0;
    int64_t pb = padded_len(n_bases, frag_len);
    return (size_t)(pb / 16 * 4 + pb / 32 * 4 + 256);
}

int mss_genome_load(const uint32_t* d_packed, const uint32_t* d_nmask, int64_t n_bases, int32_t frag_len, int32_t overlap,
                    void* d_workspace, size_t workspace_bytes, void* stream, mss_genome_t** out)
{
    if (!out) return MSS_ERR_ARG;
    *out = nullptr;
    if (!d_packed || !d_workspace || n_bases <= 0 || frag_len <= 0 || overlap < -1) return MSS_ERR_ARG;
    if (frag_len > (1 << 24)) return MSS_ERR_RANGE;
    int64_t nfrag = (n_bases + frag_len - 1) / frag_len;
    if (nfrag > 2147483647ll) return MSS_ERR_RANGE;
    if (workspace_bytes < mss_genome_workspace_bytes(n_bases, frag_len, overlap)) return MSS_ERR_WORKSPACE;
    if (((uintptr_t)d_workspace & 15) != 0) return MSS_ERR_ARG;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return cuda_fail(e);
    mss_genome* g = new (std::nothrow) mss_genome;
    if (!g) return MSS_ERR_ARG;
    int64_t pb = padded_len(n_bases, frag_len);
    uint32_t* wp = (uint32_t*)d_workspace;
    uint32_t* wn = wp + pb / 16;
    g->packed = wp; g->nmask = wn; g->n_bases = n_bases; g->padded_bases = pb;
    g->frag_len = frag_len; g->overlap = overlap; g->n_frag = (int32_t)nfrag;
    g->device = dev; g->sm_count = prop.multiProcessorCount; g->max_smem_optin = (int)prop.sharedMemPerBlockOptin;
    e = launch_genome_prepare(d_packed, d_nmask, n_bases, pb, wp, wn, (cudaStream_t)stream);
    if (e != cudaSuccess) { delete g; return cuda_fail(e); }
    *out = g;
    return MSS_OK;
}

int mss_genome_free(mss_genome_t* g)
{
    if (!g) return MSS_ERR_ARG;
    delete g;
    return MSS_OK;
}

int32_t mss_genome_num_fragments(const mss_genome_t* g) { return g ? g->n_frag : 0; }
int64_t mss_genome_num_bases(const mss_genome_t* g) { return g ? g->n_bases : 0; }

size_t mss_map_workspace_bytes(const mss_genome_t* g, int32_t n_reads, int32_t max_len, int32_t strands)
{
    if (!g || n_reads < 0 || max_len < 1 || strands < 1 || strands > 3) return 0;
    size_t a = scan_generic_workspace(g, n_reads);
    size_t b = scan_dpx_workspace(g, n_reads, max_len, strands);
    size_t c = scan_two_pass_workspace(g, n_reads, strands);
    if (b > a) a = b;
    return c > a ? c : a;
}

static int map_reads_impl(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                          const int32_t* d_lens, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t strands,
                          void* d_workspace, size_t workspace_bytes, void* stream, mss_top2_t* d_out,
                          int32_t istep, const uint32_t* d_pssm, int32_t pssm_stride)
{
    if (!g || n_reads < 0 || strands < 1 || strands > 3 || max_len < 1) return MSS_ERR_ARG;
    if (n_reads == 0) return MSS_OK;
    if (!d_reads || !d_lens || !d_out || !d_workspace) return MSS_ERR_ARG;
    if ((int64_t)read_stride_words * 16 < max_len) return MSS_ERR_ARG;
    int rc = check_scoring_scan(sc, max_len);
    if (rc != MSS_OK) return rc;
    if ((rc = check_device(g)) != MSS_OK) return rc;
    if (workspace_bytes < mss_map_workspace_bytes(g, n_reads, max_len, strands)) return MSS_ERR_WORKSPACE;
    ScanParams p;
    p.gpacked = g->packed; p.gnmask = g->nmask; p.n_bases = g->n_bases;
    p.F = g->frag_len; p.V = g->overlap; p.n_frag = g->n_frag;
    p.reads = d_reads; p.reads_nmask = d_reads_nmask; p.stride_words = read_stride_words; p.lens = d_lens;
    p.n_reads = n_reads; p.max_len = max_len; p.match = sc.match; p.mismatch = sc.mismatch; p.strands = strands; p.zero = 0;
    p.istep = istep; p.pssm = d_pssm; p.pssm_stride = pssm_stride; p.ubound = nullptr; p.delta = 0;
    cudaError_t e;
    bool use_generic = (t_variant == 1) || !scan_dpx_supported(g, p);
    bool two_pass = !use_generic && (t_variant == 0 || t_variant == 7) && scan_filter_supported(g, p);   // 2..6: one-pass tiles
    if (use_generic) e = launch_scan_generic(g, p, d_workspace, workspace_bytes, d_out, (cudaStream_t)stream, &t_info);
    else if (two_pass) e = launch_scan_two_pass(g, p, d_workspace, workspace_bytes, d_out, (cudaStream_t)stream, &t_info);
    else e = launch_scan_dpx(g, p, d_workspace, workspace_bytes, d_out, (cudaStream_t)stream, &t_info, t_variant);
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

int mss_map_reads(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                  const int32_t* d_lens, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t strands,
                  void* d_workspace, size_t workspace_bytes, void* stream, mss_top2_t* d_out)
{
    return map_reads_impl(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, sc, strands, d_workspace,
                          workspace_bytes, stream, d_out, 1, nullptr, 0);
}

int mss_map_reads_fast(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                       const int32_t* d_lens, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t strands,
                       void* d_workspace, size_t workspace_bytes, void* stream, mss_top2_t* d_out)
{
    return map_reads_impl(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, sc, strands, d_workspace,
                          workspace_bytes, stream, d_out, 2, nullptr, 0);
}

static int bounds_impl(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                       const int32_t* d_lens, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t strands,
                       int32_t every_other, void* stream, uint16_t* d_bounds, int32_t* h_delta,
                       const uint32_t* d_pssm, int32_t pssm_stride)
{
    if (!g || n_reads < 0 || strands < 1 || strands > 3 || max_len < 1) return MSS_ERR_ARG;
    if (h_delta) *h_delta = 0;
    if (n_reads == 0) return MSS_OK;
    if (!d_reads || !d_lens || !d_bounds) return MSS_ERR_ARG;
    if ((int64_t)read_stride_words * 16 < max_len) return MSS_ERR_ARG;
    int rc = check_scoring_scan(sc, max_len);
    if (rc != MSS_OK) return rc;
    if ((rc = check_device(g)) != MSS_OK) return rc;
    ScanParams p;
    p.gpacked = g->packed; p.gnmask = g->nmask; p.n_bases = g->n_bases;
    p.F = g->frag_len; p.V = g->overlap; p.n_frag = g->n_frag;
    p.reads = d_reads; p.reads_nmask = d_reads_nmask; p.stride_words = read_stride_words; p.lens = d_lens;
    p.n_reads = n_reads; p.max_len = max_len; p.match = sc.match; p.mismatch = sc.mismatch; p.strands = strands; p.zero = 0;
    p.istep = every_other ? 2 : 1; p.pssm = d_pssm; p.pssm_stride = pssm_stride; p.ubound = nullptr; p.delta = 0;
    if (!scan_filter_supported(g, p)) return MSS_ERR_RANGE;
    if (h_delta) *h_delta = scan_filter_delta(p);
    cudaError_t e = launch_scan_filter(g, p, d_bounds, (cudaStream_t)stream, nullptr, nullptr, nullptr, nullptr, nullptr);
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

int mss_map_reads_bounds(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                         const int32_t* d_lens, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t strands,
                         int32_t every_other, void* stream, uint16_t* d_bounds, int32_t* h_delta)
{
    return bounds_impl(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, sc, strands, every_other, stream,
                       d_bounds, h_delta, nullptr, 0);
}

int mss_map_reads_bounds_pssm(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                              const int32_t* d_lens, int32_t n_reads, int32_t max_len, const uint32_t* d_pssm, int32_t pssm_stride,
                              mss_scoring_t bound, int32_t strands, void* stream, uint16_t* d_bounds, int32_t* h_delta)
{
    if (n_reads > 0 && (!d_pssm || pssm_stride < max_len)) return MSS_ERR_ARG;
    return bounds_impl(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, bound, strands, 0, stream,
                       d_bounds, h_delta, d_pssm, pssm_stride);
}

int mss_pssm_build(const uint8_t* d_qual, int32_t qual_stride, const int32_t* d_lens, int32_t n_reads, mss_scoring_t sc,
                   int32_t scale, void* stream, uint32_t* d_pssm, int32_t pssm_stride)
{
    if (n_reads < 0 || qual_stride < 1 || pssm_stride < 1 || scale < 1) return MSS_ERR_ARG;
    if (n_reads == 0) return MSS_OK;
    if (!d_qual || !d_lens || !d_pssm) return MSS_ERR_ARG;
    if (sc.match <= 0 || sc.mismatch >= 0) return MSS_ERR_RANGE;
    if ((int64_t)scale * sc.match > 32767 || (int64_t)scale * sc.mismatch < -32768) return MSS_ERR_RANGE;
    // phred Q -> x = P(base correct) = 1 - 10^(-Q/10); match*x and mismatch*x/3 in fixed point, decided
    // in IEEE double on the host (94 values), rounded to nearest with halves away from zero
    PssmLut lut;
    for (int q = 0; q < 94; q++) {
        double x = 1.0 - pow(10.0, -(double)q / 10.0);
        long long pm = llround((double)scale * (double)sc.match * x);
        long long px = llround((double)scale * (double)sc.mismatch * x / 3.0);
        lut.v[q] = ((uint32_t)(uint16_t)(int16_t)pm) | ((uint32_t)(uint16_t)(int16_t)px << 16);
    }
    cudaError_t e = launch_pssm_build(d_qual, qual_stride, d_lens, n_reads, lut, (cudaStream_t)stream, d_pssm, pssm_stride);
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

int mss_map_reads_pssm(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                       const int32_t* d_lens, int32_t n_reads, int32_t max_len, const uint32_t* d_pssm, int32_t pssm_stride,
                       mss_scoring_t bound, int32_t strands, void* d_workspace, size_t workspace_bytes, void* stream,
                       mss_top2_t* d_out)
{
    if (n_reads > 0 && (!d_pssm || pssm_stride < max_len)) return MSS_ERR_ARG;
    return map_reads_impl(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, bound, strands, d_workspace,
                          workspace_bytes, stream, d_out, 1, d_pssm, pssm_stride);
}

size_t mss_map_host_workspace_bytes(const mss_genome_t* g, int32_t n_reads, int32_t max_len, int32_t read_stride_words,
                                    int32_t strands)
{
    size_t base = mss_map_workspace_bytes(g, n_reads, max_len, strands);
    if (base == 0 || read_stride_words < 1) return 0;
    size_t n = (size_t)(n_reads > 0 ? n_reads : 1);
    size_t reads = (n * read_stride_words * 4 + 255) / 256 * 256;
    size_t mask = (n * ((read_stride_words + 1) / 2) * 4 + 255) / 256 * 256;
    size_t lens = (n * 4 + 255) / 256 * 256;
    size_t outb = (n * sizeof(mss_top2_t) + 255) / 256 * 256;
    return (base + 255) / 256 * 256 + reads + mask + lens + outb;
}

int mss_map_reads_host(const mss_genome_t* g, const uint32_t* h_reads, const uint32_t* h_reads_nmask, int32_t read_stride_words,
                       const int32_t* h_lens, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t strands,
                       void* d_workspace, size_t workspace_bytes, void* stream, mss_top2_t* h_out)
{
    if (!g || n_reads < 0 || read_stride_words < 1) return MSS_ERR_ARG;
    if (n_reads == 0) return MSS_OK;
    if (!h_reads || !h_lens || !h_out || !d_workspace) return MSS_ERR_ARG;
    size_t need = mss_map_host_workspace_bytes(g, n_reads, max_len, read_stride_words, strands);
    if (need == 0) return MSS_ERR_ARG;
    if (workspace_bytes < need) return MSS_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    size_t n = (size_t)n_reads;
    size_t base = (mss_map_workspace_bytes(g, n_reads, max_len, strands) + 255) / 256 * 256;
    size_t reads_b = n * read_stride_words * 4, mask_b = n * ((read_stride_words + 1) / 2) * 4, lens_b = n * 4;
    char* w = (char*)d_workspace;
    uint32_t* d_reads = (uint32_t*)(w + base);
    uint32_t* d_mask = (uint32_t*)((char*)d_reads + (reads_b + 255) / 256 * 256);
    int32_t* d_lens = (int32_t*)((char*)d_mask + (mask_b + 255) / 256 * 256);
    mss_top2_t* d_out = (mss_top2_t*)((char*)d_lens + (lens_b + 255) / 256 * 256);
    cudaError_t e = cudaMemcpyAsync(d_reads, h_reads, reads_b, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && h_reads_nmask) e = cudaMemcpyAsync(d_mask, h_reads_nmask, mask_b, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_lens, h_lens, lens_b, cudaMemcpyHostToDevice, st);
    // from here on copies from / to the caller's host buffers may be in flight: no return without a synchronise
    if (e != cudaSuccess) { cudaStreamSynchronize(st); return cuda_fail(e); }
    int rc = mss_map_reads(g, d_reads, h_reads_nmask ? d_mask : nullptr, read_stride_words, d_lens, n_reads, max_len, sc,
                           strands, d_workspace, base, st, d_out);
    if (rc != MSS_OK) { cudaStreamSynchronize(st); return rc; }
    e = cudaMemcpyAsync(h_out, d_out, n * sizeof(mss_top2_t), cudaMemcpyDeviceToHost, st);
    cudaError_t es = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = es;
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

size_t mss_nw_workspace_bytes(const mss_genome_t* g, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t pad)
{
    if (!g || n_reads < 0 || max_len < 1 || pad < 0 || sc.match <= 0 || sc.mismatch >= 0 || sc.gap >= 0) return 0;
    return nw_workspace(g, n_reads, max_len, sc, pad);
}

static int nw_align_impl(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                 const int32_t* d_lens, int32_t n_reads, int32_t max_len, const mss_top2_t* d_hits, mss_scoring_t sc,
                 int32_t pad, void* d_workspace, size_t workspace_bytes, void* stream,
                 int32_t* d_score, int64_t* d_ref_pos, uint32_t* d_cigar, int32_t cigar_stride, int32_t* d_n_cigar,
                 const uint32_t* d_pssm, int32_t pssm_stride)
{
    if (!g || n_reads < 0 || max_len < 1 || pad < 0 || cigar_stride < 1) return MSS_ERR_ARG;
    if (n_reads == 0) return MSS_OK;
    if (!d_reads || !d_lens || !d_hits || !d_score || !d_ref_pos || !d_cigar || !d_n_cigar || !d_workspace) return MSS_ERR_ARG;
    if ((int64_t)read_stride_words * 16 < max_len) return MSS_ERR_ARG;
    if (sc.match <= 0 || sc.mismatch >= 0 || sc.gap >= 0) return MSS_ERR_RANGE;
    if (max_len > MSS_MAX_READ_LEN) return MSS_ERR_RANGE;
    if ((int64_t)max_len * (int64_t)(-sc.gap) > (1ll << 30) || (int64_t)max_len * sc.match > (1ll << 30)) return MSS_ERR_RANGE;
    if (workspace_bytes < mss_nw_workspace_bytes(g, n_reads, max_len, sc, pad)) return MSS_ERR_WORKSPACE;
    int rcd = check_device(g);
    if (rcd != MSS_OK) return rcd;
    cudaError_t e = launch_nw(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, d_hits, d_pssm, pssm_stride,
                              sc, pad, d_workspace, workspace_bytes, (cudaStream_t)stream, d_score, d_ref_pos, d_cigar,
                              cigar_stride, d_n_cigar);
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

int mss_nw_align(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                 const int32_t* d_lens, int32_t n_reads, int32_t max_len, const mss_top2_t* d_hits, mss_scoring_t sc,
                 int32_t pad, void* d_workspace, size_t workspace_bytes, void* stream,
                 int32_t* d_score, int64_t* d_ref_pos, uint32_t* d_cigar, int32_t cigar_stride, int32_t* d_n_cigar)
{
    return nw_align_impl(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, d_hits, sc, pad, d_workspace,
                         workspace_bytes, stream, d_score, d_ref_pos, d_cigar, cigar_stride, d_n_cigar, nullptr, 0);
}

int mss_nw_align_pssm(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                      const int32_t* d_lens, int32_t n_reads, int32_t max_len, const mss_top2_t* d_hits,
                      const uint32_t* d_pssm, int32_t pssm_stride, mss_scoring_t bound, int32_t pad,
                      void* d_workspace, size_t workspace_bytes, void* stream,
                      int32_t* d_score, int64_t* d_ref_pos, uint32_t* d_cigar, int32_t cigar_stride, int32_t* d_n_cigar)
{
    if (n_reads > 0 && (!d_pssm || pssm_stride < max_len)) return MSS_ERR_ARG;
    return nw_align_impl(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, d_hits, bound, pad, d_workspace,
                         workspace_bytes, stream, d_score, d_ref_pos, d_cigar, cigar_stride, d_n_cigar, d_pssm, pssm_stride);
}

namespace {
inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }
}

size_t mss_map_align_host_workspace_bytes(const mss_genome_t* g, int32_t n_reads, int32_t max_len, int32_t read_stride_words,
                                          int32_t strands, mss_scoring_t sc, int32_t pad, int32_t cigar_stride)
{
    size_t a = mss_map_workspace_bytes(g, n_reads, max_len, strands);
    size_t b = mss_nw_workspace_bytes(g, n_reads, max_len, sc, pad);
    if (a == 0 || b == 0 || read_stride_words < 1 || cigar_stride < 1) return 0;
    size_t n = (size_t)(n_reads > 0 ? n_reads : 1);
    size_t scratch = up256(a > b ? a : b);
    return scratch + up256(n * read_stride_words * 4) + up256(n * ((read_stride_words + 1) / 2) * 4) + up256(n * 4)
         + up256(n * sizeof(mss_top2_t)) + up256(n * 4) + up256(n * 8) + up256(n * (size_t)cigar_stride * 4) + up256(n * 4);
}

int mss_map_align_host(const mss_genome_t* g, const uint32_t* h_reads, const uint32_t* h_reads_nmask, int32_t read_stride_words,
                       const int32_t* h_lens, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t strands, int32_t pad,
                       void* d_workspace, size_t workspace_bytes, void* stream, mss_top2_t* h_top2, int32_t* h_score,
                       int64_t* h_ref_pos, uint32_t* h_cigar, int32_t cigar_stride, int32_t* h_n_cigar)
{
    if (!g || n_reads < 0 || read_stride_words < 1 || cigar_stride < 1) return MSS_ERR_ARG;
    if (n_reads == 0) return MSS_OK;
    if (!h_reads || !h_lens || !h_top2 || !h_score || !h_ref_pos || !h_cigar || !h_n_cigar || !d_workspace) return MSS_ERR_ARG;
    size_t need = mss_map_align_host_workspace_bytes(g, n_reads, max_len, read_stride_words, strands, sc, pad, cigar_stride);
    if (need == 0) return MSS_ERR_ARG;
    if (workspace_bytes < need) return MSS_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    size_t n = (size_t)n_reads;
    size_t a = mss_map_workspace_bytes(g, n_reads, max_len, strands), b = mss_nw_workspace_bytes(g, n_reads, max_len, sc, pad);
    size_t scratch = up256(a > b ? a : b);
    size_t reads_b = n * read_stride_words * 4, mask_b = n * ((read_stride_words + 1) / 2) * 4;
    char* w = (char*)d_workspace + scratch;
    uint32_t* d_reads = (uint32_t*)w;            w += up256(reads_b);
    uint32_t* d_mask = (uint32_t*)w;             w += up256(mask_b);
    int32_t* d_lens = (int32_t*)w;               w += up256(n * 4);
    mss_top2_t* d_top2 = (mss_top2_t*)w;         w += up256(n * sizeof(mss_top2_t));
    int32_t* d_score = (int32_t*)w;              w += up256(n * 4);
    int64_t* d_pos = (int64_t*)w;                w += up256(n * 8);
    uint32_t* d_cigar = (uint32_t*)w;            w += up256(n * (size_t)cigar_stride * 4);
    int32_t* d_ncig = (int32_t*)w;
    cudaError_t e = cudaMemcpyAsync(d_reads, h_reads, reads_b, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && h_reads_nmask) e = cudaMemcpyAsync(d_mask, h_reads_nmask, mask_b, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_lens, h_lens, n * 4, cudaMemcpyHostToDevice, st);
    // from here on copies from / to the caller's host buffers may be in flight: no return without a synchronise
    if (e != cudaSuccess) { cudaStreamSynchronize(st); return cuda_fail(e); }
    const uint32_t* dm = h_reads_nmask ? d_mask : nullptr;
    int rc = mss_map_reads(g, d_reads, dm, read_stride_words, d_lens, n_reads, max_len, sc, strands, d_workspace, scratch, st, d_top2);
    if (rc != MSS_OK) { cudaStreamSynchronize(st); return rc; }
    rc = mss_nw_align(g, d_reads, dm, read_stride_words, d_lens, n_reads, max_len, d_top2, sc, pad, d_workspace, scratch, st,
                      d_score, d_pos, d_cigar, cigar_stride, d_ncig);
    if (rc != MSS_OK) { cudaStreamSynchronize(st); return rc; }
    e = cudaMemcpyAsync(h_top2, d_top2, n * sizeof(mss_top2_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_score, d_score, n * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_ref_pos, d_pos, n * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_cigar, d_cigar, n * (size_t)cigar_stride * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_n_cigar, d_ncig, n * 4, cudaMemcpyDeviceToHost, st);
    cudaError_t es = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = es;
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

int mss_mapq_filter(const mss_top2_t* d_hits, int32_t n_reads, double mapq_threshold, void* stream, uint8_t* d_mapped, float* d_mapq)
{
    if (n_reads < 0) return MSS_ERR_ARG;
    if (n_reads == 0) return MSS_OK;
    if (!d_hits || !d_mapped) return MSS_ERR_ARG;
    cudaError_t e = launch_mapq(d_hits, n_reads, mapq_threshold, (cudaStream_t)stream, d_mapped, d_mapq);
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

const char* mss_strerror(int status)
{
    switch (status) {
        case MSS_OK: return "ok";
        case MSS_ERR_ARG: return "invalid argument";
        case MSS_ERR_RANGE: return "value outside the supported range (scores, read length or fragment geometry)";
        case MSS_ERR_WORKSPACE: return "workspace too small";
        case MSS_ERR_CUDA: return "CUDA error (see mss_last_cuda_error)";
        case MSS_ERR_STATIC_LIMIT: return "the request needs more scratch than the library's built-in static buffer (mss_static_scratch_bytes): use mss_map_reads with a caller workspace";
        default: return "unknown status";
    }
}

int mss_last_cuda_error(void) { return t_last_cuda; }
int mss_version(void) { return 100; }

int mss_set_scan_variant(int variant)
{
    if (variant < 0 || variant > 13) return MSS_ERR_ARG;
    // 7: the two-pass scan, pass 1 picks its kernel and tile; 8..12: pass 1 = the tile kernel of scan_filter.cu with one tile
    // geometry forced; 13: the tile kernel with its own choice of tile (tuning and cross-checks)
    scan_filter_force_variant(variant >= 8 && variant <= 12 ? variant - 8 : -1, variant >= 8);
    if (variant >= 8) variant = 7;
    t_variant = variant;
    return MSS_OK;
}

int mss_set_pass1_geometry(int32_t query_sets, int32_t tile_window_starts, int32_t arithmetic)
{
    if (!(query_sets == 0 || query_sets == 1 || query_sets == 2 || query_sets == 4)) return MSS_ERR_ARG;
    if (tile_window_starts < 0 || (tile_window_starts & 1)) return MSS_ERR_ARG;
    if (!(arithmetic == -1 || (arithmetic >= 0 && arithmetic <= 2) || (arithmetic >= 8 && arithmetic <= 11) ||
          (arithmetic >= 16 && arithmetic <= 19) || (arithmetic >= 32 && arithmetic <= 35))) return MSS_ERR_ARG;
    scan_filter_lq_tune(query_sets, tile_window_starts / 2, arithmetic);
    return MSS_OK;
}

int mss_set_two_pass_chunk_bytes(int64_t bytes) { scan_set_two_pass_chunk_bytes(bytes); return MSS_OK; }

int mss_set_pass_timing(int on) { scan_set_pass_timing(on != 0); return MSS_OK; }

int mss_get_pass_times(float* h_pass1_ms, float* h_pass2_ms)
{
    if (!h_pass1_ms || !h_pass2_ms) return MSS_ERR_ARG;
    cudaError_t e = scan_get_pass_times(h_pass1_ms, h_pass2_ms);
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

int mss_get_last_launch(mss_launch_info_t* out)
{
    if (!out) return MSS_ERR_ARG;
    *out = t_info;
    return MSS_OK;
}

int mss_probe_dpx_peak(int32_t iters, void* stream, double* h_instr_per_s, float* h_ms)
{
    if (iters < 1 || !h_instr_per_s || !h_ms) return MSS_ERR_ARG;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(e);
    e = run_dpx_probe(iters, (cudaStream_t)stream, sms, h_instr_per_s, h_ms);
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

int mss_probe_pipe(int32_t which, int32_t iters, void* stream, double* h_per_clk_sm)
{
    if (which < 0 || which >= MSS_PROBE_COUNT || iters < 1 || !h_per_clk_sm) return MSS_ERR_ARG;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(e);
    e = run_pipe_probe(which, iters, (cudaStream_t)stream, sms, h_per_clk_sm);
    if (e != cudaSuccess) return cuda_fail(e);
    return MSS_OK;
}

}  // extern "C"
