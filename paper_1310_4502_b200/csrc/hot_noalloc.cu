// hot_noalloc.cu -- ONE entry point that allocates nothing: hot_sort_keys_noalloc, the stable radix sort of S2
// (hot_build.cu: launch_radix_sort, unchanged) with its scratch -- digit counts, their scans, tile tickets and the two
// look-back state arrays -- in a file-scope device array instead of the library's pooled cudaMalloc buffers.
// For callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
//
//   * The array is sized for HOT_NOALLOC_MAX_N keys (2^22: 2.1 MB); every GPU that loads the library holds it until exit.
//   * In host code `g_sort_scratch` is a host-side stand-in, not a device address: its device address is taken once per
//     device with cudaGetSymbolAddress (device current) and that pointer goes to the kernels.
//   * Every call shares the array, which keeps the last call's contents: the part a sort reads before writing is cleared
//     at the start of every call (stream-ordered).  Calls that overlap on the GPU (two streams) race on it.
//   * No cudaMalloc, cudaFree, or allocating library routine is called here or in launch_radix_sort.
#include <cstdio>

#include "hot_internal.h"

#define HOT_NOALLOC_MAX_N (1ll << 22)
// sort_hist_elems(2^22) = 4352 + 2 * 256 * 1024 words (hot_build.cu: SORT_STATE0 + two state arrays of 256 words per 4096-key tile)
#define HOT_NOALLOC_SCRATCH_WORDS (4352 + 2 * 256 * 1024)

static __device__ __align__(256) uint32_t g_sort_scratch[HOT_NOALLOC_SCRATCH_WORDS];

namespace {
char g_na_err[256] = "";
uint32_t* g_scratch_ptr[64] = {}; // device address of g_sort_scratch, per device
int na_fail(int code, const char* msg) {
    snprintf(g_na_err, sizeof(g_na_err), "%s", msg);
    return code;
}
} // namespace

// the eight 8-bit digit histograms of the keys (what keygen_kernel counts on the library's own path), into hist[8][256]
__global__ void __launch_bounds__(256) noalloc_hist_kernel(const uint64_t* __restrict__ key, int64_t n, uint32_t* __restrict__ hist) {
    __shared__ uint32_t h[8][256];
#pragma unroll
    for (int p = 0; p < 8; ++p) h[p][threadIdx.x] = 0;
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t k = key[i];
#pragma unroll
        for (int p = 0; p < 8; ++p) atomicAdd(&h[p][(uint32_t)(k >> (8 * p)) & 255u], 1u);
    }
    __syncthreads();
#pragma unroll
    for (int p = 0; p < 8; ++p) { const uint32_t c = h[p][threadIdx.x]; if (c) atomicAdd(&hist[p * 256 + threadIdx.x], c); }
}

extern "C" {

const char* hot_noalloc_last_error(void) { return g_na_err; }

int hot_sort_keys_noalloc(uint64_t* key, uint32_t* perm, uint64_t* key_work, uint32_t* idx_work, int64_t n, void* cuda_stream) {
    if (!key || !perm || !key_work || !idx_work) return na_fail(HOT_EINVAL, "hot_sort_keys_noalloc: NULL argument");
    if (n < 1) return na_fail(HOT_EINVAL, "hot_sort_keys_noalloc: n must be >= 1");
    if (n > HOT_NOALLOC_MAX_N) {
        snprintf(g_na_err, sizeof(g_na_err), "hot_sort_keys_noalloc: n = %lld exceeds the fixed scratch of %lld keys (2^22); use hot_build",
                 (long long)n, (long long)HOT_NOALLOC_MAX_N);
        return HOT_EINVAL;
    }
    if (sort_hist_elems(n) > (size_t)HOT_NOALLOC_SCRATCH_WORDS) return na_fail(HOT_EINTERNAL, "hot_sort_keys_noalloc: scratch layout changed");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return na_fail(HOT_ECUDA, "hot_sort_keys_noalloc: cudaGetDevice failed"); }
    if (!g_scratch_ptr[dev]) { // once per device, with that device current
        uint32_t* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_sort_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            snprintf(g_na_err, sizeof(g_na_err), "hot_sort_keys_noalloc: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
            return HOT_ECUDA;
        }
        g_scratch_ptr[dev] = p;
    }
    uint32_t* const hist = g_scratch_ptr[dev];
    // the scratch keeps the last call's contents: counts, scans, tickets and both look-back arrays of this size start at zero
    cudaError_t e = cudaMemsetAsync(hist, 0, sort_hist_elems(n) * sizeof(uint32_t), st);
    if (e == cudaSuccess) {
        int64_t nb = (n + 256 * 16 - 1) / (256 * 16);
        if (nb > 148 * 8) nb = 148 * 8;
        HOT_LAUNCHED(1);
        noalloc_hist_kernel<<<(unsigned)nb, 256, 0, st>>>(key, n, hist);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        uint64_t* kk[2] = {key, key_work};
        uint32_t* ii[2] = {perm, idx_work};
        e = launch_radix_sort(kk, ii, n, hist, st); // eight passes: the result is back in key / perm
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        snprintf(g_na_err, sizeof(g_na_err), "hot_sort_keys_noalloc: %s", cudaGetErrorString(e));
        return HOT_ECUDA;
    }
    return HOT_OK;
}

} // extern "C"
