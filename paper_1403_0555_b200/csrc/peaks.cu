// peaks.cu -- roofline denominators measured on the device in use (not part of the method):
// FP64 FMA issue rate (the bound of the resident relaxation kernels) and conflict-free
// 128-bit shared-memory load bandwidth (their co-limit).
#include "u1gf_internal.h"

namespace u1gf {
namespace {

constexpr int kChains = 8;

__global__ void __launch_bounds__(512) dfma_kernel(double* out, int iters, double a, double b) {
    double x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = (double)(threadIdx.x + c) * 1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int c = 0; c < kChains; ++c) x[c] = fma(x[c], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;  // never true; keeps the chains alive
}

// FP64 FMA streams whose multiplicands are REGISTERS, as they are in the neighbour sum w_i (link x gauge value +
// accumulator): PATTERN 1 = three distinct register operands per DFMA, nothing reusable; PATTERN 2 = the complex
// multiply-accumulate of the kernels, (ux,gx,wr)(ux,gy,wi)(uy,gy,wr)(-uy,gx,wi).  On B200 these issue at 3 and
// about 2.75 cycles per scheduler instead of the 2 of the constant-operand stream above: the register file
// delivers two 64-bit operands per issue slot pair, the third costs a cycle.
template <int PATTERN>
__global__ void __launch_bounds__(512) dfma_reg_kernel(const double* __restrict__ in, double* out, int iters) {
    double p[8], q[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        p[j] = in[threadIdx.x + 512 * j];
        q[j] = in[threadIdx.x + 512 * (8 + j)];
    }
    double a0 = p[0], a1 = p[1], a2 = p[2], a3 = p[3];
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (PATTERN == 1) {
                a0 = fma(p[j], q[j], a0);
                a1 = fma(p[(j + 1) & 7], q[(j + 3) & 7], a1);
                a2 = fma(p[(j + 2) & 7], q[(j + 5) & 7], a2);
                a3 = fma(p[(j + 3) & 7], q[(j + 7) & 7], a3);
            } else {
                const int j2 = (j + 1) & 7;
                a0 = fma(p[j], q[j], a0);
                a1 = fma(p[j], q[j2], a1);
                a0 = fma(p[j2], q[j2], a0);
                a1 = fma(-p[j2], q[j], a1);
            }
        }
    }
    const double s = a0 + a1 + a2 + a3;
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;  // never true for the zero-filled input
}

__global__ void __launch_bounds__(512) lds_kernel(unsigned* out, int iters) {
    extern __shared__ uint4 buf[];
    const int n = 8 * blockDim.x;
    for (int i = threadIdx.x; i < n; i += blockDim.x) buf[i] = make_uint4(i, i + 1, i + 2, i + 3);
    __syncthreads();
    uint4 acc = make_uint4(0, 0, 0, 0);
    int idx = threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint4 v = buf[idx + u * blockDim.x];  // consecutive lanes -> consecutive 16 B: conflict free
            acc.x ^= v.x;
            acc.y ^= v.y;
            acc.z ^= v.z;
            acc.w ^= v.w;
        }
        idx = threadIdx.x + (acc.x == 0xdeadbeefu ? 1 : 0);  // opaque dependence; the address does not change
    }
    if ((acc.x ^ acc.y ^ acc.z ^ acc.w) == 0x12345u) out[blockIdx.x * blockDim.x + threadIdx.x] = acc.x;
}

}  // namespace
}  // namespace u1gf

using namespace u1gf;

extern "C" {

int u1gf_measure_fp64_peak(double ms, double* dfma_per_s, void* cuda_stream) {
    t_launches = 0;
    if (!dfma_per_s || !(ms > 0.0)) return fail(U1GF_EINVAL, "u1gf_measure_fp64_peak: bad argument");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    double* scratch = nullptr;
    const int threads = 512, blocks = sms * 4;
    U1GF_CUDA(cudaMalloc(&scratch, (size_t)threads * blocks * sizeof(double)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 4096;
    const double per_launch = (double)threads * blocks * (double)iters * 4.0 * kChains;
    double best = 0.0, spent = 0.0;
    dfma_kernel<<<blocks, threads, 0, st>>>(scratch, iters, 0.999999, 1e-9);  // warm-up
    ++t_launches;
    while (spent < ms) {
        cudaEventRecord(e0, st);
        dfma_kernel<<<blocks, threads, 0, st>>>(scratch, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, st);
        ++t_launches;
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) {
            cudaFree(scratch);
            return fail(U1GF_ECUDA, "u1gf_measure_fp64_peak: %s", cudaGetErrorString(e));
        }
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        spent += t;
        const double rate = per_launch / (t * 1e-3);
        if (rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(scratch);
    *dfma_per_s = best;
    return U1GF_OK;
}

int u1gf_measure_fp64_rate(int32_t pattern, double ms, double* dfma_per_s, void* cuda_stream) {
    if (pattern == 0) return u1gf_measure_fp64_peak(ms, dfma_per_s, cuda_stream);
    t_launches = 0;
    if (!dfma_per_s || !(ms > 0.0) || pattern < 0 || pattern > 2)
        return fail(U1GF_EINVAL, "u1gf_measure_fp64_rate: bad argument");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int threads = 512, blocks = sms * 2, iters = 8192;
    double *in = nullptr, *scratch = nullptr;
    U1GF_CUDA(cudaMalloc(&in, (size_t)threads * 16 * sizeof(double)));
    U1GF_CUDA(cudaMalloc(&scratch, (size_t)threads * blocks * sizeof(double)));
    U1GF_CUDA(cudaMemsetAsync(in, 0, (size_t)threads * 16 * sizeof(double), st));
    auto kern = pattern == 1 ? dfma_reg_kernel<1> : dfma_reg_kernel<2>;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const double per_launch = (double)threads * blocks * (double)iters * 8.0 * 4.0;
    double best = 0.0, spent = 0.0;
    kern<<<blocks, threads, 0, st>>>(in, scratch, 16);  // warm-up
    ++t_launches;
    cudaError_t e = cudaSuccess;
    while (spent < ms) {
        cudaEventRecord(e0, st);
        kern<<<blocks, threads, 0, st>>>(in, scratch, iters);
        cudaEventRecord(e1, st);
        ++t_launches;
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        spent += t;
        const double rate = per_launch / (t * 1e-3);
        if (rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(in);
    cudaFree(scratch);
    if (e != cudaSuccess) return fail(U1GF_ECUDA, "u1gf_measure_fp64_rate: %s", cudaGetErrorString(e));
    *dfma_per_s = best;
    return U1GF_OK;
}

int u1gf_measure_smem_peak(double ms, double* bytes_per_s, void* cuda_stream) {
    t_launches = 0;
    if (!bytes_per_s || !(ms > 0.0)) return fail(U1GF_EINVAL, "u1gf_measure_smem_peak: bad argument");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    unsigned* scratch = nullptr;
    const int threads = 512, blocks = sms * 2;
    const size_t smem = ((size_t)8 * threads + 1) * sizeof(uint4);
    U1GF_CUDA(cudaFuncSetAttribute(lds_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    U1GF_CUDA(cudaMalloc(&scratch, (size_t)threads * blocks * sizeof(unsigned)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 4096;
    const double per_launch = (double)threads * blocks * (double)iters * 8.0 * 16.0;
    double best = 0.0, spent = 0.0;
    lds_kernel<<<blocks, threads, smem, st>>>(scratch, iters);
    ++t_launches;
    while (spent < ms) {
        cudaEventRecord(e0, st);
        lds_kernel<<<blocks, threads, smem, st>>>(scratch, iters);
        cudaEventRecord(e1, st);
        ++t_launches;
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) {
            cudaFree(scratch);
            return fail(U1GF_ECUDA, "u1gf_measure_smem_peak: %s", cudaGetErrorString(e));
        }
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        spent += t;
        const double rate = per_launch / (t * 1e-3);
        if (rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(scratch);
    *bytes_per_s = best;
    return U1GF_OK;
}

}  // extern "C"
