// a0 genome load: pad to nfrag*F (+ look-ahead room) with N; derived device layout.
#include "mss_common.cuh"

__global__ void genome_prepare_kernel(const uint32_t* __restrict__ in_packed, const uint32_t* __restrict__ in_nmask,
                                      int64_t n_bases, int64_t padded_bases,
                                      uint32_t* __restrict__ out_packed, uint32_t* __restrict__ out_nmask)
{
    int64_t n_pw = padded_bases / 16, n_mw = padded_bases / 32;
    int64_t in_pw = (n_bases + 15) / 16, in_mw = (n_bases + 31) / 32;
    for (int64_t w = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; w < n_pw; w += (int64_t)gridDim.x * blockDim.x) {
        uint32_t v = w < in_pw ? in_packed[w] : 0u;
        int64_t first = w * 16;
        if (first + 16 > n_bases) {                       // clear codes beyond the end (they are N anyway)
            int64_t keep = n_bases - first;
            v = keep <= 0 ? 0u : (v & ((keep >= 16) ? 0xFFFFFFFFu : ((1u << (2 * keep)) - 1u)));
        }
        out_packed[w] = v;
    }
    for (int64_t w = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; w < n_mw; w += (int64_t)gridDim.x * blockDim.x) {
        uint32_t v = (in_nmask && w < in_mw) ? in_nmask[w] : 0u;
        int64_t first = w * 32;
        if (first + 32 > n_bases) {                       // every position >= n_bases is N
            int64_t keep = n_bases - first;
            uint32_t valid = keep <= 0 ? 0u : ((keep >= 32) ? 0xFFFFFFFFu : ((1u << keep) - 1u));
            v = (v & valid) | ~valid;
        }
        out_nmask[w] = v;
    }
}

cudaError_t launch_genome_prepare(const uint32_t* d_packed, const uint32_t* d_nmask, int64_t n_bases,
                                  int64_t padded_bases, uint32_t* out_packed, uint32_t* out_nmask, cudaStream_t st)
{
    int64_t words = padded_bases / 16;
    int blocks = (int)((words + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    genome_prepare_kernel<<<blocks, 256, 0, st>>>(d_packed, d_nmask, n_bases, padded_bases, out_packed, out_nmask);
    return cudaGetLastError();
}
