// Repeat filter / MAPQ on the top-2 records and the live DPX issue-rate probe.
#include <math_constants.h>
#include "mss_common.cuh"

// Decisions and the logarithm are taken in IEEE double (this file's --use_fast_math only touches single precision): the
// default (thr < 0) is the paper's "ratio below .9" on the integers; a threshold >= 0 is a MAPQ cutoff.
__global__ void mapq_kernel(const mss_top2_t* __restrict__ hits, int32_t n, double thr, uint8_t* __restrict__ mapped,
                            float* __restrict__ mapq)
{
    int32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    mss_top2_t t = hits[r];
    double q = 0.0;
    uint8_t ok = 0;
    if (t.best.frag >= 0 && t.best.score > 0) {                            // else: ratio undefined -> unmapped, MAPQ 0
        int32_t second = (t.second.frag >= 0) ? t.second.score : 0;
        if (second <= 0) q = CUDART_INF;                                    // p = 0: nothing competes
        else q = -100.0 * log2((double)second / (double)t.best.score);
        if (thr < 0.0) ok = (10ll * second < 9ll * t.best.score) ? 1 : 0;
        else ok = (q > thr) ? 1 : 0;
    }
    mapped[r] = ok;
    if (mapq) mapq[r] = (float)q;
}

cudaError_t launch_mapq(const mss_top2_t* d_hits, int32_t n_reads, double thr, cudaStream_t st, uint8_t* d_mapped, float* d_mapq)
{
    mapq_kernel<<<(n_reads + 255) / 256, 256, 0, st>>>(d_hits, n_reads, thr, d_mapped, d_mapq);
    return cudaGetLastError();
}

// Base qualities -> per-position (pmatch, pmismatch) table rows: a 94-entry lookup of the phred value
// (values above 93, the FASTQ maximum, count as 93); positions at or beyond len[r] get (0, 0).
__global__ void pssm_build_kernel(const uint8_t* __restrict__ qual, int32_t qual_stride, const int32_t* __restrict__ lens,
                                  int32_t n_reads, PssmLut lut, uint32_t* __restrict__ pssm, int32_t pssm_stride)
{
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (int64_t)n_reads * pssm_stride) return;
    int32_t r = (int32_t)(idx / pssm_stride), i = (int32_t)(idx % pssm_stride);
    uint32_t v = 0u;
    if (i < lens[r] && i < qual_stride) {
        uint32_t q = qual[(int64_t)r * qual_stride + i];
        v = lut.v[q > 93u ? 93u : q];
    }
    pssm[idx] = v;
}

cudaError_t launch_pssm_build(const uint8_t* d_qual, int32_t qual_stride, const int32_t* d_lens, int32_t n_reads,
                              const PssmLut& lut, cudaStream_t st, uint32_t* d_pssm, int32_t pssm_stride)
{
    int64_t total = (int64_t)n_reads * pssm_stride;
    pssm_build_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(d_qual, qual_stride, d_lens, n_reads, lut, d_pssm, pssm_stride);
    return cudaGetLastError();
}

// 8 independent chains per thread, per round: 8 VIADDMNMX.S16x2.RELU + 4 VIMNMX3.S16x2 (the scan's own 2:1 mix)
__global__ void __launch_bounds__(1024) dpx_probe_kernel(uint32_t* out, uint32_t a, uint32_t b, int iters)
{
    uint32_t h[8], m[4];
#pragma unroll
    for (int j = 0; j < 8; j++) h[j] = a * (threadIdx.x + j + 1);
#pragma unroll
    for (int j = 0; j < 4; j++) m[j] = 0;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < 4; u++) {
#pragma unroll
            for (int j = 0; j < 8; j++) h[j] = __viaddmax_s16x2_relu(h[j], h[(j + 1) & 7], b);
#pragma unroll
            for (int j = 0; j < 4; j++) m[j] = __vimax3_s16x2(m[j], h[2 * j], h[2 * j + 1]);
        }
    }
    uint32_t s = 0;
#pragma unroll
    for (int j = 0; j < 4; j++) s ^= m[j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

cudaError_t run_dpx_probe(int32_t iters, cudaStream_t st, int sm_count, double* instr_per_s, float* ms)
{
    uint32_t* out = nullptr;
    int blocks = sm_count * 2;
    cudaError_t e = cudaMalloc(&out, (size_t)blocks * 1024 * 4);   // probe only: not on the mapping path
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    dpx_probe_kernel<<<blocks, 1024, 0, st>>>(out, 0x00010003u, 0u, iters / 8 + 1);
    cudaEventRecord(e0, st);
    dpx_probe_kernel<<<blocks, 1024, 0, st>>>(out, 0x00010003u, 0u, iters);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) {
        cudaEventElapsedTime(ms, e0, e1);
        *instr_per_s = (double)blocks * 1024.0 * (double)iters * 48.0 / ((double)*ms * 1e-3);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return e == cudaSuccess ? cudaGetLastError() : e;
}


// ---- issue-rate probes behind the roofline denominators ---------------------------------------------
// 8 independent register chains per thread, 1024 threads x 1 block per SM; thread-instructions (row 4: cells) per clock per
// SM from clock64() around the loop.  Operands vary per thread so that nothing is promoted to the uniform datapath.
// Rows: 0 VIADDMNMX.S16x2.RELU, 1 VIMNMX3.S16x2, 2 their 2:1 mix, 3 LDS.32 conflict-free, 4 the exact scan's inner mix.
namespace {
template <int WHICH>
__global__ void __launch_bounds__(1024) pipe_probe_kernel(uint32_t* out, long long* cyc, uint32_t a, uint32_t b, uint32_t c, int iters)
{
    __shared__ uint32_t sm[8192];
    uint32_t h[8], m[8];
    { uint32_t lz; asm volatile("mov.u32 %0, %%laneid;" : "=r"(lz)); lz >>= 5; a += lz; b += lz; c += lz; }   // opaque, per-thread
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) sm[i] = a * i;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 8; j++) { h[j] = a * (threadIdx.x + j + 1); m[j] = b + j + threadIdx.x * 0x00070005u; }
    const uint32_t* myp = sm + threadIdx.x;
    long long t0 = clock64();
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
#pragma unroll
            for (int j = 0; j < 8; j++) {
                if (WHICH == 0) h[j] = __viaddmax_s16x2_relu(h[j], m[j], c);
                if (WHICH == 1) h[j] = __vimax3_s16x2(h[j], m[j], c);
                if (WHICH == 2) { h[j] = __viaddmax_s16x2_relu(h[j], m[j], c); if (j & 1) m[j] = __vimax3_s16x2(m[j], h[j], h[j - 1]); }
                if (WHICH == 3) {   // LDS.32 only (conflict-free), one LOP3 consumer each
                    uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(myp + ((u * 8 + j) & 63) * 32 + (it & 1) * 2048)));
                    h[j] ^= v;
                }
                if (WHICH == 4) {   // the exact scan's inner mix: LDS.32 + VIADDMNMX.S16x2.RELU per 2 cells, VIMNMX3.S16x2 per 4 cells
                    uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(myp + ((u * 8 + j) & 63) * 32 + (it & 1) * 2048)));
                    uint32_t hn = __viaddmax_s16x2_relu(h[j], v, c);
                    if (u & 1) m[j] = __vimax3_s16x2(m[j], h[j], hn);
                    h[j] = hn;
                }
            }
        }
    }
    long long t1 = clock64();
    uint32_t s = 0;
#pragma unroll
    for (int j = 0; j < 8; j++) s ^= h[j] ^ m[j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

const double kProbeCount[MSS_PROBE_COUNT] = { 1, 1, 1.5, 1, 2 };   // counted units per chain step (row 4: cells)

template <int WHICH>
cudaError_t launch_pipe_probe(uint32_t* out, long long* cyc, int blocks, int iters, cudaStream_t st)
{
    pipe_probe_kernel<WHICH><<<blocks, 1024, 0, st>>>(out, cyc, 0x00010003u, 0x00020001u, 0u, iters);
    return cudaGetLastError();
}
}  // namespace

cudaError_t run_pipe_probe(int which, int32_t iters, cudaStream_t st, int sm_count, double* per_clk_sm)
{
    if (which < 0 || which >= MSS_PROBE_COUNT) return cudaErrorInvalidValue;
    uint32_t* out = nullptr; long long* cyc = nullptr;
    int blocks = sm_count;
    cudaError_t e = cudaMalloc(&out, (size_t)blocks * 1024 * 4);                 // probe only: not on the mapping path
    if (e == cudaSuccess) e = cudaMalloc(&cyc, (size_t)blocks * 8);
    if (e != cudaSuccess) { cudaFree(out); return e; }
    for (int pass = 0; pass < 2 && e == cudaSuccess; pass++) {                   // pass 0 warms up
        switch (which) {
            case 0: e = launch_pipe_probe<0>(out, cyc, blocks, iters, st); break;
            case 1: e = launch_pipe_probe<1>(out, cyc, blocks, iters, st); break;
            case 2: e = launch_pipe_probe<2>(out, cyc, blocks, iters, st); break;
            case 3: e = launch_pipe_probe<3>(out, cyc, blocks, iters, st); break;
            default: e = launch_pipe_probe<4>(out, cyc, blocks, iters, st); break;
        }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) {
        long long* h = new long long[blocks];
        e = cudaMemcpy(h, cyc, (size_t)blocks * 8, cudaMemcpyDeviceToHost);
        double avg = 0;
        for (int i = 0; i < blocks; i++) avg += (double)h[i];
        avg /= blocks;
        delete[] h;
        *per_clk_sm = (double)iters * 64.0 * kProbeCount[which] * 1024.0 / avg;
    }
    cudaFree(out); cudaFree(cyc);
    return e;
}
