// mss_map_reads_static: mss_map_reads for callers that cannot allocate or hand over device scratch (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc).  The scan's scratch -- the 16-bit pass-1 bounds of the
// two-pass scan, or the partial top-2 records of the one-pass / generic scan -- lives in a file-scope device array of
// MSS_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.  The entry point calls no
// cudaMalloc, cudaFree or allocating library routine; the kernels are the ones mss_map_reads launches, given this array as
// their workspace.
//
// In host code the array's name is only a host-side stand-in for the symbol, not a device address: a kernel handed it would
// fault (or silently use the wrong memory where the GPU can reach host memory).  The device address is looked up here, in the
// array's own translation unit, once per device and with that device current, by cudaGetSymbolAddress.
#include <mutex>
#include "mss_common.cuh"

namespace {

static __device__ __align__(256) unsigned char g_static_scratch[MSS_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
void* g_scratch_ptr[kMaxDevices] = { nullptr };        // device address of g_static_scratch on device d (nullptr = not looked up)
std::mutex g_scratch_mutex;

// the array's address on the CURRENT device; looked up on first use per device
int static_scratch(void** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return mss_record_cuda_error(e);
    if (dev < 0 || dev >= kMaxDevices) return MSS_ERR_RANGE;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) return mss_record_cuda_error(e != cudaSuccess ? e : cudaErrorInvalidSymbol);
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return MSS_OK;
}

}  // namespace

extern "C" {

size_t mss_static_scratch_bytes(void) { return (size_t)MSS_STATIC_SCRATCH_BYTES; }

int mss_static_init(void)
{
    void* p = nullptr;
    return static_scratch(&p);
}

int mss_map_reads_static(const mss_genome_t* g, const uint32_t* d_reads, const uint32_t* d_reads_nmask, int32_t read_stride_words,
                         const int32_t* d_lens, int32_t n_reads, int32_t max_len, mss_scoring_t sc, int32_t strands,
                         void* stream, mss_top2_t* d_out)
{
    if (!g || n_reads < 0 || strands < 1 || strands > 3 || max_len < 1) return MSS_ERR_ARG;
    if (n_reads == 0) return MSS_OK;
    const size_t need = mss_map_workspace_bytes(g, n_reads, max_len, strands);
    if (need == 0) return MSS_ERR_ARG;
    if (need > (size_t)MSS_STATIC_SCRATCH_BYTES) return MSS_ERR_STATIC_LIMIT;      // the batch is too large for the built-in buffer
    void* scratch = nullptr;
    int rc = static_scratch(&scratch);          // the handle's device must be current (mss_map_reads checks it again)
    if (rc != MSS_OK) return rc;
    // Nothing in the scratch has to start at zero: pass 1 writes every bound before pass 2 reads it, and the one-pass / generic
    // scans write every partial record before the merge reads it, so the previous call's contents are simply overwritten.
    return mss_map_reads(g, d_reads, d_reads_nmask, read_stride_words, d_lens, n_reads, max_len, sc, strands, scratch,
                         (size_t)MSS_STATIC_SCRATCH_BYTES, stream, d_out);
}

}  // extern "C"
