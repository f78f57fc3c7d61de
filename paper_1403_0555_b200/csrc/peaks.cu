// peaks.cu -- libu1gf_measure.so: roofline denominators measured on the device in use (not part of the method):
// FP64 FMA issue rate (the bound of the resident relaxation kernels) and conflict-free
// 128-bit shared-memory load bandwidth (their co-limit).
#include "../../include/u1gf_measure.h"
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

// PATTERN 3 / 4: the reusable-operand stream / the three-fresh-operand stream with two independent integer
// instructions per DFMA: on B200 the integer work does NOT hide behind the FP64 pipe (2.26 -> 3.4 and 3.0 -> 4.8 cycles
// per DFMA per scheduler), i.e. every instruction of the relaxation kernel counts.
template <int FRESH>
__global__ void __launch_bounds__(512) dfma_int_kernel(const double* __restrict__ in, double* out, unsigned* iout, int iters,
                                                       unsigned m) {
    double g[8], u[8], acc[8];
    unsigned x[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        g[c] = in[threadIdx.x + 512 * c];
        u[c] = in[threadIdx.x + 512 * (8 + c)];
        acc[c] = in[threadIdx.x + c];
        x[c] = threadIdx.x * (c + 1);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                if (FRESH) acc[c] = fma(u[(c + r) & 7], g[c], acc[c]);
                else acc[c] = fma(u[r], g[r], acc[c]);
                x[c] = (x[c] ^ m) + x[(c + 3) & 7];
            }
    }
    double s = 0;
    unsigned xs = 0;
#pragma unroll
    for (int c = 0; c < 8; ++c) s += acc[c], xs ^= x[c];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (xs == 0x1234567u) iout[threadIdx.x] = xs;
}

// PATTERN 5: one dependent DFMA chain per warp, one warp per scheduler: the reported rate is 32 x 4 x 148 / latency.
__global__ void __launch_bounds__(128) dfma_chain_kernel(double* out, int iters, double a, double b) {
    double x = threadIdx.x * 1e-3;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 32; ++u) x = fma(x, a, b);
    }
    if (x == 123.456) out[threadIdx.x] = x;
}

// PATTERN 6: FP64 tensor-core MMA (DMMA m8n8k4, 8 FMAs per thread and instruction): the same pipe as DFMA on B200, at
// 2.0 cycles per 32 FMAs per scheduler -- the neighbour sum is a sparse stencil, densifying it would double its flops.
__global__ void __launch_bounds__(512) dmma_kernel(const double* __restrict__ in, double* out, int iters) {
    double a[4], b[4], c[8][2];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        a[j] = in[threadIdx.x + 512 * j];
        b[j] = in[threadIdx.x + 512 * (4 + j)];
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) c[j][0] = c[j][1] = 0.0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int j = 0; j < 8; ++j)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[j][0]), "+d"(c[j][1])
                             : "d"(a[r]), "d"(b[(r + j) & 3]));
    }
    double s = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += c[j][0] + c[j][1];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
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

// Shared-memory instruction mixes: NL warp-uniform LDS.128 (a link: every lane the same address), NG lane-strided
// LDS.128 (a neighbour of 32 starts: 512 contiguous bytes), NS lane-strided STS.128, per "site"; 8 sites per iteration.
template <int NL, int NG, int NS>
__global__ void __launch_bounds__(512) lds_mix_kernel(unsigned* out, int iters) {
    extern __shared__ uint4 buf[];   // 96 KB
    for (int i = threadIdx.x; i < 6144; i += blockDim.x) buf[i] = make_uint4(i, i + 1, i + 2, i + 3);
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint4 acc = make_uint4(0, 0, 0, 0);
    int lb = warp * 64;
    const int gb = 1024 + lane, sb = 1024 + warp * 32 + lane;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int s = 0; s < 8; ++s) {
#pragma unroll
            for (int j = 0; j < NL; ++j) {
                const uint4 v = buf[lb + s * 8 + j];
                acc.x ^= v.x; acc.y ^= v.y; acc.z ^= v.z; acc.w ^= v.w;
            }
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                const uint4 v = buf[gb + ((s * 4 + j + warp) & 15) * 32 * 8 + s * 32];
                acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
            }
#pragma unroll
            for (int j = 0; j < NS; ++j) buf[sb + (s + 8 * j) * 512 % 5120] = acc;
        }
        lb += (acc.x == 0xdeadbeefu);   // opaque dependence; the address does not change
    }
    if ((acc.x ^ acc.y) == 0x12345u) out[threadIdx.x] = acc.x;
}

// Distributed shared memory (thread-block clusters): every CTA of a cluster of `csize` CTAs (512 threads, 200 KB of
// shared memory, one CTA per SM -- the footprint of a resident relaxation kernel) pulls 512-byte rows, one 128-bit word
// per lane, out of the shared memory of its neighbour in the cluster (REMOTE) or out of its own through the cluster
// window.  This is the halo exchange a cluster-resident kernel for 6^4 / 8^4 would live on.
__device__ __forceinline__ unsigned dsmem_mapa(unsigned addr, unsigned rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
template <bool REMOTE>
__global__ void __launch_bounds__(512) dsmem_kernel(double* out, int iters, int csize) {
    extern __shared__ __align__(16) double2 dsm[];
    unsigned rank;
    asm("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    for (int i = threadIdx.x; i < 12800; i += blockDim.x) dsm[i] = make_double2((double)i, (double)rank);
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;\n");
    const unsigned base = (unsigned)__cvta_generic_to_shared(dsm);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned ra = dsmem_mapa(base + (warp * 8 * 32 + lane) * 16, REMOTE ? (rank + 1) % (unsigned)csize : rank);
    double acc = 0.0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int h = 0; h < 8; ++h) {
            double2 v;
            asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(ra + h * 512 + ((it * 37) & 15) * 4096));
            acc += v.x + v.y;
        }
    }
    if (acc == 1.2345) out[0] = acc;   // never true; keeps the loads alive
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;\n");
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
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaFree(scratch);
        return fail(U1GF_ECUDA, "cudaEventCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
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
    if (!dfma_per_s || !(ms > 0.0) || pattern < 0 || pattern > 6)
        return fail(U1GF_EINVAL, "u1gf_measure_fp64_rate: bad argument");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int threads = pattern == 5 ? 128 : 512, blocks = pattern == 5 ? sms : sms * 2, iters = pattern == 5 ? 2048 : 8192;
    double *in = nullptr, *scratch = nullptr;
    U1GF_CUDA(cudaMalloc(&in, (size_t)threads * 16 * sizeof(double)));
    U1GF_CUDA(cudaMalloc(&scratch, (size_t)threads * blocks * sizeof(double)));
    U1GF_CUDA(cudaMemsetAsync(in, 0, (size_t)threads * 16 * sizeof(double), st));
    unsigned* iscratch = nullptr;
    if (pattern == 3 || pattern == 4) U1GF_CUDA(cudaMalloc(&iscratch, (size_t)threads * sizeof(unsigned)));
    auto run = [&](int it) {
        switch (pattern) {
            case 1: dfma_reg_kernel<1><<<blocks, threads, 0, st>>>(in, scratch, it); break;
            case 2: dfma_reg_kernel<2><<<blocks, threads, 0, st>>>(in, scratch, it); break;
            case 3: dfma_int_kernel<0><<<blocks, threads, 0, st>>>(in, scratch, iscratch, it, 5u); break;
            case 4: dfma_int_kernel<1><<<blocks, threads, 0, st>>>(in, scratch, iscratch, it, 5u); break;
            case 5: dfma_chain_kernel<<<blocks, threads, 0, st>>>(scratch, it, 0.999999, 1e-9); break;
            default: dmma_kernel<<<blocks, threads, 0, st>>>(in, scratch, it); break;
        }
    };
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaFree(scratch);
        return fail(U1GF_ECUDA, "cudaEventCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    // thread-level FMAs per launch: 32 per iteration, except the DMMA stream (32 instructions x 8 FMAs)
    const double per_launch = (double)threads * blocks * (double)iters * 32.0 * (pattern == 6 ? 8.0 : 1.0);
    double best = 0.0, spent = 0.0;
    run(16);  // warm-up
    ++t_launches;
    cudaError_t e = cudaSuccess;
    while (spent < ms) {
        cudaEventRecord(e0, st);
        run(iters);
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
    if (iscratch) cudaFree(iscratch);
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
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaFree(scratch);
        return fail(U1GF_ECUDA, "cudaEventCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
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

int u1gf_measure_smem_rate(int32_t mix, double ms, double* instr_per_s, void* cuda_stream) {
    t_launches = 0;
    if (!instr_per_s || !(ms > 0.0) || mix < 0 || mix > 2) return fail(U1GF_EINVAL, "u1gf_measure_smem_rate: bad argument");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int threads = 512, blocks = sms, iters = 2048;
    const size_t smem = 98304;
    void (*kern)(unsigned*, int) = mix == 0 ? lds_mix_kernel<0, 4, 1> : mix == 1 ? lds_mix_kernel<8, 0, 0> : lds_mix_kernel<8, 4, 1>;
    const double per_site = mix == 0 ? 5.0 : mix == 1 ? 8.0 : 13.0;
    U1GF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    unsigned* scratch = nullptr;
    U1GF_CUDA(cudaMalloc(&scratch, (size_t)threads * sizeof(unsigned)));
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaFree(scratch);
        return fail(U1GF_ECUDA, "cudaEventCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    const double per_launch = (double)(threads / 32) * blocks * (double)iters * 8.0 * per_site;   // warp-level instructions
    double best = 0.0, spent = 0.0;
    kern<<<blocks, threads, smem, st>>>(scratch, 16);
    ++t_launches;
    cudaError_t e = cudaSuccess;
    while (spent < ms) {
        cudaEventRecord(e0, st);
        kern<<<blocks, threads, smem, st>>>(scratch, iters);
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
    cudaFree(scratch);
    if (e != cudaSuccess) return fail(U1GF_ECUDA, "u1gf_measure_smem_rate: %s", cudaGetErrorString(e));
    *instr_per_s = best;
    return U1GF_OK;
}

int u1gf_measure_dsmem_rate(int32_t cluster_size, int32_t remote, double ms, double* bytes_per_s_per_sm,
                            int32_t* max_active_clusters, void* cuda_stream) {
    t_launches = 0;
    if (!bytes_per_s_per_sm || !max_active_clusters || !(ms > 0.0) || cluster_size < 1 || cluster_size > 16)
        return fail(U1GF_EINVAL, "u1gf_measure_dsmem_rate: bad argument");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    auto kern = remote ? dsmem_kernel<true> : dsmem_kernel<false>;
    const int smem = 200 * 1024;
    U1GF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    U1GF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(512);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)cluster_size;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cfg.gridDim = dim3((unsigned)cluster_size);
    int ncl = 0;
    U1GF_CUDA(cudaOccupancyMaxActiveClusters(&ncl, kern, &cfg));
    *max_active_clusters = ncl;
    *bytes_per_s_per_sm = 0.0;
    if (ncl < 1) return U1GF_OK;
    cfg.gridDim = dim3((unsigned)(cluster_size * ncl));
    double* scratch = nullptr;
    U1GF_CUDA(cudaMalloc(&scratch, 64));
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaFree(scratch);
        return fail(U1GF_ECUDA, "cudaEventCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    const int iters = 4000;
    const double per_cta = (double)iters * 8.0 * 512.0 * 16.0;   // 16 warps x 8 loads x 512 bytes per iteration
    double best = 0.0, spent = 0.0;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, scratch, 50, (int)cluster_size);   // warm-up
    ++t_launches;
    while (e == cudaSuccess && spent < ms) {
        cudaEventRecord(e0, st);
        e = cudaLaunchKernelEx(&cfg, kern, scratch, iters, (int)cluster_size);
        cudaEventRecord(e1, st);
        ++t_launches;
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        spent += t;
        const double rate = per_cta / (t * 1e-3);
        if (rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(scratch);
    if (e != cudaSuccess) return fail(U1GF_ECUDA, "u1gf_measure_dsmem_rate: %s", cudaGetErrorString(e));
    *bytes_per_s_per_sm = best;
    return U1GF_OK;
}

}  // extern "C"
