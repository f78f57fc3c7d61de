// discovery.cu -- SURVEY section 8(f) item 1: what the paper reads off its sorted functional values.
//   * u1gf_discovery_curve: number of distinct copies found within the first 2^k samples, k = 0, 1, ... -- the curves
//     of PAPER.md Figs. 1-3 ("number of minima as a function of the number of samples", L149).  Copies are numbered
//     in order of first discovery by u1gf_count_copies, so the curve is a cumulative histogram of the bit length of
//     each copy's first position.
//   * u1gf_paper_count: the paper's own estimate of the number of copies, the number of distinct integers
//     X = floor(x * 1e8), x = 1 - F/(dV), among the converged samples -- for comparison with the
//     tolerance clustering of u1gf_count_copies (reading R7: 1e-8 keys can merge distinct copies and split one copy
//     at a key boundary).
// Integer work only; no floating-point atomics.
#include <cub/device/device_radix_sort.cuh>

#include <mutex>

#include "u1gf_internal.h"

namespace u1gf {
namespace {

constexpr unsigned long long kNoKey = ~0ull;

__global__ void __launch_bounds__(1024) curve_kernel(unsigned long long n_distinct, const long long* __restrict__ rep,
                                                     int n_levels, long long* __restrict__ curve) {
    __shared__ unsigned long long hist[66];   // hist[b] = copies whose first position has bit length b (0 for position 0)
    for (int b = threadIdx.x; b < 66; b += blockDim.x) hist[b] = 0ull;
    __syncthreads();
    for (unsigned long long c = threadIdx.x; c < n_distinct; c += blockDim.x) {
        const unsigned long long p = (unsigned long long)rep[c];
        atomicAdd(&hist[64 - __clzll((long long)p)], 1ull);   // p < 2^k  <=>  bit length of p <= k
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long run = 0ull;
        for (int k = 0; k < n_levels; ++k) {
            if (k <= 64) run += hist[k];
            curve[k] = (long long)run;
        }
    }
}

__global__ void paper_keys_kernel(unsigned long long n, const double* __restrict__ F_norm, const uint8_t* __restrict__ status,
                                  double scale, unsigned long long* __restrict__ keys) {
    const unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    unsigned long long key = kNoKey;
    if ((status[i] & 1u) == 0u) {
        const double x = __dmul_rn(__dsub_rn(1.0, F_norm[i]), scale);   // x * 1e8 exactly as written (no contraction)
        const long long X = (long long)floor(x);
        key = (unsigned long long)(X + (1ll << 62));   // order preserving, never the sentinel
    }
    keys[i] = key;
}

__global__ void count_runs_kernel(unsigned long long n, const unsigned long long* __restrict__ keys,
                                  unsigned long long* __restrict__ n_keys) {
    const unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x;
    int first = 0;
    if (i < n && keys[i] != kNoKey) first = (i == 0 || keys[i - 1] != keys[i]) ? 1 : 0;
    const unsigned m = __ballot_sync(0xffffffffu, first);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(n_keys, (unsigned long long)__popc(m));
}

size_t sort_temp_bytes(uint64_t n) {
    size_t t = 0;
    cub::DeviceRadixSort::SortKeys(nullptr, t, (const unsigned long long*)nullptr, (unsigned long long*)nullptr,
                                   (unsigned long long)n);
    return (t + 255) & ~(size_t)255;
}

}  // namespace
}  // namespace u1gf

// ---------------------------------------------------------------------------------------------------------------------
// Scratch for u1gf_paper_count_static (see include/u1gf.h).  The array is part of this library's device image: each GPU
// on which this file's device code gets loaded keeps kStaticScratchBytes of it until the process exits, used or not.
// Layout during a call: keys [n] | sorted keys [n] | CUB sort temporary -- the layout u1gf_paper_count puts in the
// caller's workspace.  Nothing in it has to be zero when a call starts: both key arrays are overwritten in full for
// i < n before they are read, and the sort zeroes the counters it keeps in its temporary itself.  The only value that
// must start at zero is the caller's n_keys, which the entry point clears on the stream.
//
// `g_static_scratch` written in HOST code is the host-side shadow of the symbol, not where the array lives on the GPU;
// static_scratch_address() asks the runtime for the real address once per device and keeps it.
// ---------------------------------------------------------------------------------------------------------------------
static constexpr size_t kStaticMaxN = (size_t)U1GF_PAPER_COUNT_STATIC_MAX_N;
// 2 key arrays of kStaticMaxN 8-byte keys (16 MiB) + the sort's temporary, a third key array plus its digit counters
// (tests/test_zz_no_alloc.py runs the full kStaticMaxN on the GPU, so a sort that wanted more would be caught).  32 MiB.
static constexpr size_t kStaticScratchBytes = 4 * kStaticMaxN * sizeof(unsigned long long);
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

namespace u1gf {
namespace {

constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
void* g_static_address[kMaxDevices] = {};   // device address of g_static_scratch on device k, NULL = not looked up yet

// Device address of the array on the CURRENT device.  The first call per device is the set-up: cudaGetSymbolAddress may
// have to load this file's device code onto that GPU, which is when the array comes into existence there.
int static_scratch_address(void** out) {
    int dev = -1;
    U1GF_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices)
        return fail(U1GF_EINVAL, "u1gf_paper_count_static: device ordinal %d outside 0..%d", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_address[dev]) {
        void* p = nullptr;
        U1GF_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return fail(U1GF_ECUDA, "u1gf_paper_count_static: cudaGetSymbolAddress returned a NULL address on device %d", dev);
        g_static_address[dev] = p;
    }
    *out = g_static_address[dev];
    return U1GF_OK;
}

}  // namespace
}  // namespace u1gf

using namespace u1gf;

extern "C" {

int u1gf_discovery_curve(uint64_t n_distinct, const int64_t* rep, int32_t n_levels, int64_t* curve, void* cuda_stream) {
    t_launches = 0;
    if (n_levels < 1 || n_levels > 65 || !curve) return fail(U1GF_EINVAL, "u1gf_discovery_curve: bad n_levels or NULL curve");
    if (n_distinct && !rep) return fail(U1GF_EINVAL, "u1gf_discovery_curve: NULL rep");
    if (int rc = check_device()) return rc;
    curve_kernel<<<1, 1024, 0, (cudaStream_t)cuda_stream>>>((unsigned long long)n_distinct, (const long long*)rep, n_levels,
                                                             (long long*)curve);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    return U1GF_OK;
}

size_t u1gf_paper_count_workspace_bytes(uint64_t n) {
    const size_t keys = (((size_t)n * 8) + 255) & ~(size_t)255;
    return 2 * keys + sort_temp_bytes(n ? n : 1) + 256;
}

int u1gf_paper_count(uint64_t n, const double* F_norm, const uint8_t* status, double scale, int64_t* n_keys,
                     void* workspace, size_t workspace_bytes, void* cuda_stream) {
    t_launches = 0;
    if (!n_keys) return fail(U1GF_EINVAL, "u1gf_paper_count: NULL n_keys");
    if (!(scale > 0.0)) return fail(U1GF_EINVAL, "u1gf_paper_count: scale must be > 0");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    U1GF_CUDA(cudaMemsetAsync(n_keys, 0, sizeof(int64_t), st));
    if (n == 0) return U1GF_OK;
    if (!F_norm || !status) return fail(U1GF_EINVAL, "u1gf_paper_count: NULL input array");
    const size_t need = u1gf_paper_count_workspace_bytes(n);
    if (!workspace || workspace_bytes < need)
        return fail(U1GF_ENOMEM, "u1gf_paper_count: workspace of %zu bytes needed, %zu given", need, workspace_bytes);
    if (((uintptr_t)workspace & 255) != 0) return fail(U1GF_EINVAL, "u1gf_paper_count: workspace not 256-byte aligned");
    const size_t kb = (((size_t)n * 8) + 255) & ~(size_t)255;
    unsigned long long* k0 = (unsigned long long*)workspace;
    unsigned long long* k1 = (unsigned long long*)((char*)workspace + kb);
    void* temp = (char*)workspace + 2 * kb;
    size_t tb = sort_temp_bytes(n);
    const unsigned blocks = (unsigned)((n + 255) / 256);
    paper_keys_kernel<<<blocks, 256, 0, st>>>((unsigned long long)n, F_norm, status, scale, k0);
    U1GF_CUDA(cudaGetLastError());
    U1GF_CUDA(cub::DeviceRadixSort::SortKeys(temp, tb, k0, k1, (unsigned long long)n, 0, 64, st));
    count_runs_kernel<<<blocks, 256, 0, st>>>((unsigned long long)n, k1, (unsigned long long*)n_keys);
    U1GF_CUDA(cudaGetLastError());
    t_launches += 2;   // own kernels; the CUB sort launches are library code and not counted
    return U1GF_OK;
}

// The same three steps as u1gf_paper_count (keys -> radix sort -> count run heads), with the scratch taken from
// g_static_scratch instead of a caller workspace.  No cudaMalloc / cudaFree / allocating library call on this path:
// cudaMemsetAsync, kernel launches and cub::DeviceRadixSort::SortKeys with its temporary storage handed in.
int u1gf_paper_count_static(uint64_t n, const double* F_norm, const uint8_t* status, double scale, int64_t* n_keys,
                            void* cuda_stream) {
    t_launches = 0;
    if (!n_keys) return fail(U1GF_EINVAL, "u1gf_paper_count_static: NULL n_keys");
    if (!(scale > 0.0)) return fail(U1GF_EINVAL, "u1gf_paper_count_static: scale must be > 0");
    if (n > (uint64_t)kStaticMaxN)
        return fail(U1GF_EINVAL,
                    "u1gf_paper_count_static: n = %llu exceeds U1GF_PAPER_COUNT_STATIC_MAX_N = %llu, the size the built-in "
                    "scratch array was compiled for; use u1gf_paper_count with a caller workspace for larger batches",
                    (unsigned long long)n, (unsigned long long)kStaticMaxN);
    if (n && (!F_norm || !status)) return fail(U1GF_EINVAL, "u1gf_paper_count_static: NULL input array");
    if (int rc = check_device()) return rc;
    void* scratch = nullptr;
    if (int rc = static_scratch_address(&scratch)) return rc;   // first call on this device: the set-up
    cudaStream_t st = (cudaStream_t)cuda_stream;
    U1GF_CUDA(cudaMemsetAsync(n_keys, 0, sizeof(int64_t), st));
    if (n == 0) return U1GF_OK;
    const size_t kb = (((size_t)n * 8) + 255) & ~(size_t)255;
    size_t tb = sort_temp_bytes(n);
    if (2 * kb + tb > kStaticScratchBytes)
        return fail(U1GF_ENOMEM, "u1gf_paper_count_static: n = %llu needs %zu bytes of scratch, the built-in array holds %zu",
                    (unsigned long long)n, 2 * kb + tb, kStaticScratchBytes);
    unsigned long long* k0 = (unsigned long long*)scratch;
    unsigned long long* k1 = (unsigned long long*)((char*)scratch + kb);
    void* temp = (char*)scratch + 2 * kb;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    paper_keys_kernel<<<blocks, 256, 0, st>>>((unsigned long long)n, F_norm, status, scale, k0);
    U1GF_CUDA(cudaGetLastError());
    U1GF_CUDA(cub::DeviceRadixSort::SortKeys(temp, tb, k0, k1, (unsigned long long)n, 0, 64, st));
    count_runs_kernel<<<blocks, 256, 0, st>>>((unsigned long long)n, k1, (unsigned long long*)n_keys);
    U1GF_CUDA(cudaGetLastError());
    t_launches += 2;
    return U1GF_OK;
}

}  // extern "C"
