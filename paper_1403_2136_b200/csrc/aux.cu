// Repeat filter / MAPQ on the top-2 records and the live DPX issue-rate probe.
#include "mss_common.cuh"

__global__ void mapq_kernel(const mss_top2_t* __restrict__ hits, int32_t n, float thr, uint8_t* __restrict__ mapped,
                            float* __restrict__ mapq)
{
    int32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    mss_top2_t t = hits[r];
    float q = 0.0f;
    uint8_t ok = 0;
    if (t.best.frag >= 0 && t.best.score > 0) {
        int32_t second = (t.second.frag >= 0) ? t.second.score : 0;
        if (second <= 0) q = 3.4e38f;
        else q = -100.0f * log2f((float)second / (float)t.best.score);
        if (thr < 0.0f) ok = (10ll * second < 9ll * t.best.score) ? 1 : 0;   // the paper's 0.9 ratio, exact integers
        else ok = (q > thr) ? 1 : 0;
    }
    mapped[r] = ok;
    if (mapq) mapq[r] = q;
}

cudaError_t launch_mapq(const mss_top2_t* d_hits, int32_t n_reads, float thr, cudaStream_t st, uint8_t* d_mapped, float* d_mapq)
{
    mapq_kernel<<<(n_reads + 255) / 256, 256, 0, st>>>(d_hits, n_reads, thr, d_mapped, d_mapq);
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
