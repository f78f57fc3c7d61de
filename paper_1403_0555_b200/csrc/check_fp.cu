// check_fp.cu -- a7 first-Gribov-region test: lowest non-trivial eigenvalue of the Faddeev-Popov operator.
// PAPER.md:L38 defines M_FP as the Hessian of the gauge-fixing functional, L9/L50 the first Gribov region as the
// set where it is positive (semi)definite; the constant vector is its exact zero mode (global gauge freedom,
// PAPER.md:L65).  The paper never evaluates M_FP; north_star asks for lambda_1 per copy by batched Lanczos.
//
// One CTA per configuration.  Shared memory holds the link weights c_{i,mu} = Re(g_i U_{i,mu} conj g_{i+mu}) and
// two Lanczos vectors; the three-term recurrence runs on the orthogonal complement of the constant vector
// (re-projected every step).  The smallest Ritz value comes from Sturm-count multisection by warp 0, the stop
// test from the residual bound beta_k |s_k| (last component of the Ritz vector).
#include "u1gf_internal.h"

namespace u1gf {
namespace {

constexpr int kMaxK = 512;  // Lanczos steps kept

struct FpParams {
    unsigned long long n_cfg;
    const double2* g;
    double tol_fp;
    double* lambda1;
    uint8_t* region;
    unsigned long long* n_in;
    int32_t* steps;   // Lanczos steps taken per configuration, or NULL
    const int64_t* index;   // configuration k is g[index[k]] (NULL: g[k])
};

__device__ __forceinline__ double block_sum(double a, double (*red)[32], int& buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) red[buf][warp] = a;
    __syncthreads();
    double s = 0.0;
    if (nw == 2) s = red[buf][0] + red[buf][1];   // the small lattices: one or two warps per configuration
    else if (nw == 1) s = red[buf][0];
    else
        for (int w = 0; w < nw; ++w) s += red[buf][w];
    buf ^= 1;
    return s;
}

// power of two that brings |p| back near 1 (0 and denormals: no scaling)
__device__ __forceinline__ double unit_scale(double p) {
    const int e = (__double2hiint(p) >> 20) & 0x7ff;
    return e == 0 ? 1.0 : __hiloint2double((2046 - e) << 20, 0);
}

// Number of eigenvalues of the k x k tridiagonal T_k (alpha[0..k), off-diagonal squares beta2[0..k-1)) below x: sign
// changes of the leading principal minors p_j = det(T_j - x), p_j = (alpha_j - x) p_{j-1} - beta_{j-1}^2 p_{j-2}.
// Division free (the pivot form q_j = p_j / p_{j-1} costs an FP64 division per step in a dependent chain); the pair
// is rescaled every 8 steps.
__device__ __forceinline__ int sturm_count(const double* alpha, const double* beta2, int k, double x) {
    double p0 = 1.0, p1 = alpha[0] - x;
    if (p1 == 0.0) p1 = 1e-300;
    int cnt = p1 < 0.0 ? 1 : 0;
    auto step = [&](double d, double b2) {
        double p2 = fma(d, p1, -b2 * p0);
        if (p2 == 0.0) p2 = p1 * 1e-300;   // a vanishing minor takes the sign of its predecessor: no change
        cnt += ((p2 < 0.0) != (p1 < 0.0)) ? 1 : 0;
        p0 = p1;
        p1 = p2;
    };
    int j = 1;
    for (; j + 3 < k; j += 4) {   // the shared-memory operands of four steps are fetched ahead of the dependent chain
        const double d0 = alpha[j] - x, d1 = alpha[j + 1] - x, d2 = alpha[j + 2] - x, d3 = alpha[j + 3] - x;
        const double b0 = beta2[j - 1], b1 = beta2[j], b2 = beta2[j + 1], b3 = beta2[j + 2];
        step(d0, b0);
        step(d1, b1);
        step(d2, b2);
        step(d3, b3);
        const double sc = unit_scale(p1);   // |p| grows at most by (4 d + 1)^4 per round: far from overflow
        p0 *= sc;
        p1 *= sc;
    }
    for (; j < k; ++j) step(alpha[j] - x, beta2[j - 1]);
    return cnt;
}

// Smallest eigenvalue of T_k by 33-way multisection on warp 0 (all 32 lanes call this), bracket [lo, hi].
__device__ double smallest_ritz(const double* alpha, const double* beta2, int k, double lo, double hi, double rtol) {
    const int lane = threadIdx.x & 31;
    for (int it = 0; it < 14; ++it) {
        const double h = (hi - lo) / 33.0;
        const double x = lo + h * (double)(lane + 1);
        const int c = sturm_count(alpha, beta2, k, x);
        const unsigned m = __ballot_sync(0xffffffffu, c >= 1);
        if (m == 0) {
            lo = lo + h * 32.0;
        } else {
            const int f = __ffs(m) - 1;  // first lane whose x lies above the smallest eigenvalue
            hi = lo + h * (double)(f + 1);
            lo = lo + h * (double)f;
        }
        if (hi - lo <= rtol * fmax(1.0, fmax(fabs(lo), fabs(hi)))) break;   // final: 2e-14; lambda_1 is compared at 1e-8 (R9, R16)
    }
    return 0.5 * (lo + hi);
}

// |last component| of the normalised eigenvector of T_k for (an approximation of) its smallest eigenvalue.  The
// components of that vector DECAY towards the end -- that decay is the convergence of the Ritz value -- so the
// three-term recurrence is run backwards from x_{k-1} = 1, the direction in which the wanted solution grows and
// rounding errors do not: x_{j-1} = ((lam - alpha_j) x_j - beta_j x_{j+1}) / beta_{j-1}.  (Run forwards it stalls
// near 1e-8, the stop test never fires and every configuration takes the maximum number of steps.)
__device__ double last_component(const double* alpha, const double* beta, const double* ibeta, int k, double lam) {
    double xn = 0.0, xc = 1.0, norm2 = 1.0, last = 1.0;   // x_{j+1}, x_j; `last` follows the scale of x_{k-1}
    for (int j = k - 1; j >= 1; --j) {
        const double bnext = j + 1 < k ? beta[j] : 0.0;
        double xp = fma(lam - alpha[j], xc, -bnext * xn) * ibeta[j - 1];
        norm2 = fma(xp, xp, norm2);
        if (norm2 > 1e200) {  // rescale
            xc *= 1e-100;
            xp *= 1e-100;
            last *= 1e-100;
            norm2 *= 1e-200;
        }
        xn = xc;
        xc = xp;
    }
    return fabs(last) * rsqrt(norm2);
}

// Sum of two values over the CTA, same result in every thread, fixed tree (see block_sum).
__device__ __forceinline__ void block_sum2(double& a, double& b, double (*red2)[32][2], int& buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) {
        red2[buf][warp][0] = a;
        red2[buf][warp][1] = b;
    }
    __syncthreads();
    double sa = 0.0, sb = 0.0;
    if (nw == 2) {
        sa = red2[buf][0][0] + red2[buf][1][0];
        sb = red2[buf][0][1] + red2[buf][1][1];
    } else if (nw == 1) {
        sa = red2[buf][0][0];
        sb = red2[buf][0][1];
    } else {
        for (int w = 0; w < nw; ++w) {
            sa += red2[buf][w][0];
            sb += red2[buf][w][1];
        }
    }
    a = sa;
    b = sb;
    buf ^= 1;
}

// One CTA per configuration, every thread owns up to SPT sites (i = tid, tid + T, ...).  The neighbour indices of a
// thread's sites are the same for every configuration and every step: they are read once into registers (16-bit,
// V <= 8192) instead of 2 DIM index loads per site and mat-vec.  Per Lanczos step: the mat-vec with <w, v1> (one
// reduction), w -= alpha v1 with the mean of w and its norm without the mean, sum w^2 - V mean^2, in ONE reduction, then
// the scaled vector -- three barriers per step.
template <int DIM, int SPT, int MAXT>
__global__ void __launch_bounds__(MAXT, MAXT <= 256 ? 2 : 1) lanczos_kernel(const OrbitDev D, const FpParams P) {
    extern __shared__ double sm[];
    const int V = D.V, tid = threadIdx.x, T = blockDim.x;
    double* c = sm;                 // [DIM][V]
    double* va = c + (size_t)V * DIM;  // [V]
    double* vb = va + V;            // [V]
    __shared__ double red[2][32];
    __shared__ double red2[2][32][2];
    const int kcap = min(V - 1, kMaxK);
    double* alpha = vb + V;   // Lanczos coefficients [4][kcap], behind the vectors in dynamic shared memory
    double* beta = alpha + kcap;
    double* beta2 = beta + kcap;
    double* ibeta = beta2 + kcap;
    __shared__ double s_lam, s_res;
    int buf = 0, buf2 = 0;
    const int kmax = kcap;

    unsigned short nf[SPT][DIM], nb[SPT][DIM];
#pragma unroll
    for (int s = 0; s < SPT; ++s) {
        const int i = tid + s * T;
#pragma unroll
        for (int mu = 0; mu < DIM; ++mu) {
            nf[s][mu] = i < V ? (unsigned short)__ldg(D.fwd + i * DIM + mu) : (unsigned short)0;
            nb[s][mu] = i < V ? (unsigned short)__ldg(D.bwd + i * DIM + mu) : (unsigned short)0;
        }
    }

    for (unsigned long long cfg = blockIdx.x; cfg < P.n_cfg; cfg += gridDim.x) {
        const double2* g = P.g + (P.index ? (unsigned long long)P.index[cfg] : cfg) * (unsigned long long)V;
        __syncthreads();
        // weights c_{i,mu} = Re(g_i U_{i,mu} conj g_{i+mu}), stored [mu][V]: consecutive lanes, consecutive banks
        double s1 = 0.0;
#pragma unroll
        for (int s = 0; s < SPT; ++s) {
            const int i = tid + s * T;
            if (i < V) {
                const double2 gi = g[i];
#pragma unroll
                for (int mu = 0; mu < DIM; ++mu) {
                    const double2 gj = g[nf[s][mu]], u = __ldg(D.U + i * DIM + mu);
                    const double ar = gi.x * u.x - gi.y * u.y, ai = gi.x * u.y + gi.y * u.x;
                    c[mu * V + i] = ar * gj.x + ai * gj.y;
                }
                // start vector: fixed pseudo-random values, constant mode removed, normalised (R16)
                const u32x4 r = philox((uint32_t)i, 0u, 0u, 5u, 0x52u, 0u);
                const double x = unit_interval_pm1(r.x, r.y);
                va[i] = x;
                s1 += x;
            }
        }
        s1 = block_sum(s1, red, buf);
        const double mean0 = s1 / (double)V;
        double s2 = 0.0;
#pragma unroll
        for (int s = 0; s < SPT; ++s) {
            const int i = tid + s * T;
            if (i < V) {
                const double x = va[i] - mean0;
                va[i] = x;
                s2 = fma(x, x, s2);
                vb[i] = 0.0;
            }
        }
        s2 = block_sum(s2, red, buf);
        const double inv0 = rsqrt(s2);
#pragma unroll
        for (int s = 0; s < SPT; ++s) {
            const int i = tid + s * T;
            if (i < V) va[i] *= inv0;
        }
        __syncthreads();

        double* v1 = va;  // current Lanczos vector
        double* v0 = vb;  // previous one; overwritten by the new direction
        double beta_prev = 0.0, lam = 0.0, lam_hi = 4.0 * DIM + 1.0;
        int k = 0, next_check = 16, k_prev = 0, n_checks = 0;
        double res_prev = 0.0, last_drop = 0.0;
        bool have_drop = false;
        bool done = false, unconverged = false;
        while (!done) {
            // w = M v1 - beta_prev v0 (kept in registers), alpha = <w, v1>
            double w[SPT], vi[SPT], a = 0.0;
#pragma unroll
            for (int s = 0; s < SPT; ++s) {
                const int i = tid + s * T;
                w[s] = 0.0;
                vi[s] = 0.0;
                if (i < V) {
                    vi[s] = v1[i];
                    double acc = 0.0;
#pragma unroll
                    for (int mu = 0; mu < DIM; ++mu) {
                        const int jf = nf[s][mu], jb = nb[s][mu];
                        acc = fma(c[mu * V + i], vi[s] - v1[jf], acc);
                        acc = fma(c[mu * V + jb], vi[s] - v1[jb], acc);
                    }
                    w[s] = fma(-beta_prev, v0[i], acc);
                    a = fma(w[s], vi[s], a);
                }
            }
            a = block_sum(a, red, buf);
            // w -= alpha v1; its mean (the constant mode, taken out every step) and its norm without the mean
            double sw = 0.0, sww = 0.0;
#pragma unroll
            for (int s = 0; s < SPT; ++s) {
                w[s] = fma(-a, vi[s], w[s]);
                sw += w[s];
                sww = fma(w[s], w[s], sww);
            }
            block_sum2(sw, sww, red2, buf2);
            const double mean = sw / (double)V;
            const double bb = fmax(fma(-(double)V * mean, mean, sww), 0.0);
            const double b = sqrt(bb);
            if (tid == 0) {
                alpha[k] = a;
                beta[k] = b;
                beta2[k] = bb;
                ibeta[k] = 1.0 / b;
            }
            ++k;
            const bool breakdown = b < 1e-13 * (4.0 * DIM);
            if (breakdown || k == kmax || k == next_check) {
                __syncthreads();
                if (tid < 32) {
                    // Ritz values decrease with k (interlacing): the new one lies below the last; a lower end a few
                    // times the last decrease below it is tried first (one Sturm count says whether it holds)
                    double lo_try = -(4.0 * DIM + 1.0);
                    if (have_drop) {
                        const double cand = lam - 8.0 * last_drop - 1e-9;
                        if (sturm_count(alpha, beta2, k, cand) == 0) lo_try = cand;
                    }
                    // the Ritz value to 1e-11 is enough to follow the residual; it is refined to 2e-14 once the test passes
                    double l = smallest_ritz(alpha, beta2, k, lo_try, lam_hi, 1e-11);
                    const double res = breakdown ? 0.0 : b * last_component(alpha, beta, ibeta, k, l - 1e-13);
                    if (breakdown || k == kmax || res < 1e-10) l = smallest_ritz(alpha, beta2, k, l - 2e-11 * fmax(1.0, fabs(l)), l + 2e-11 * fmax(1.0, fabs(l)), 2e-14);
                    if (tid == 0) {
                        s_lam = l;
                        s_res = res;
                    }
                }
                __syncthreads();
                if (n_checks > 0) {
                    last_drop = fmax(lam - s_lam, 0.0);
                    have_drop = true;
                }
                lam = s_lam;
                lam_hi = lam + 1e-9;
                const double res = s_res;
                if (breakdown || k == kmax || res < 1e-10) done = true;
                unconverged = !breakdown && !(res < 1e-10) && k < V - 1;   // k = V-1: the Krylov space is the whole of 1-perp, T_k is exact
                // next test where the residual bound, which falls geometrically, is expected to cross 1e-10
                int step = max(4, k / 4);
                if (n_checks > 0 && res > 0.0 && res < res_prev) {   // (a measured decay may carry the next test up to k/2 ahead)
                    const double per_step = log(res_prev / res) / (double)(k - k_prev);
                    step = max(3, min(max(4, k / 2), (int)(0.9 * log(res / 1e-10) / per_step) + 1));
                }
                res_prev = res;
                k_prev = k;
                ++n_checks;
                next_check = k + step;
            }
            if (!done) {
                const double ib = 1.0 / b;
#pragma unroll
                for (int s = 0; s < SPT; ++s) {
                    const int i = tid + s * T;
                    if (i < V) v0[i] = (w[s] - mean) * ib;   // the new vector takes the place of the one before the last
                }
                double* tmp = v0;
                v0 = v1;
                v1 = tmp;
                beta_prev = b;
                __syncthreads();
            }
        }
        if (tid == 0) {
            P.lambda1[cfg] = lam;
            const uint8_t reg = lam > P.tol_fp ? 1 : (fabs(lam) <= P.tol_fp ? 2 : 0);
            // bit 2: the step cap was reached with the residual bound still above 1e-10 (R16): lambda1 is then only an
            // upper bound of the eigenvalue and the caller should not trust a region of 1 or 2
            P.region[cfg] = (uint8_t)(reg | (unconverged ? 4 : 0));
            if (P.steps) P.steps[cfg] = k;
            if (reg) atomicAdd(P.n_in, 1ull);
        }
    }
}

template <int DIM>
int launch(const u1gf_orbit* o, const FpParams& P, cudaStream_t st) {
    const int V = o->dev.V;
    const int kcap = V - 1 < kMaxK ? V - 1 : kMaxK;
    const size_t smem = ((size_t)V * DIM + 2 * (size_t)V + 4 * (size_t)(kcap > 0 ? kcap : 1)) * sizeof(double);
    if (smem > 220 * 1024)
        return fail(U1GF_EINVAL, "u1gf_check_fp: lattice of %d sites does not fit the resident Lanczos kernel", V);
    // few threads per configuration: the Ritz test is serial work of one warp, during which the other warps of the
    // CTA wait; many small CTAs per SM keep the SM busy with other configurations meanwhile (measured: 8 warps per
    // configuration spent 54 % of their time at that barrier)
    // sites per thread: 8 for the large lattices; fewer on the small ones, where a configuration is one or two warps and
    // the SM needs more of them in flight to cover the latencies of the dependent chain of a Lanczos step (measured, hot
    // orbits: 4^4 43.1 / 35.1 / 46.6 ms per 131072 copies at 8 / 4 / 2 sites per thread, 4^3 7.9 / 4.5 / 3.8 ms per 65536)
#ifndef U1GF_FP_SPT4_MAXV
#define U1GF_FP_SPT4_MAXV 512
#endif
    const int spt = V <= 128 ? 2 : (V <= U1GF_FP_SPT4_MAXV ? 4 : 8);
    const int T = ((V + spt - 1) / spt + 31) / 32 * 32;
    // the thread count bounds the registers ptxas may use
    auto kern = spt == 8 ? (T <= 256 ? lanczos_kernel<DIM, 8, 256> : lanczos_kernel<DIM, 8, 640>)
                         : (spt == 4 ? (T <= 256 ? lanczos_kernel<DIM, 4, 256> : lanczos_kernel<DIM, 4, 640>) : lanczos_kernel<DIM, 2, 256>);
    if (T > 640) return fail(U1GF_EINVAL, "u1gf_check_fp: lattice of %d sites does not fit the resident Lanczos kernel", V);
    if (smem > 48 * 1024) U1GF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    U1GF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T, smem));
    if (per_sm < 1) return fail(U1GF_ECUDA, "u1gf_check_fp: kernel does not fit on an SM");
    unsigned long long grid = (unsigned long long)per_sm * o->sm_count;
    if (grid > P.n_cfg) grid = P.n_cfg;
    kern<<<(unsigned)grid, T, smem, st>>>(o->dev, P);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    return U1GF_OK;
}

}  // namespace
}  // namespace u1gf

using namespace u1gf;

extern "C" int u1gf_check_fp(const u1gf_orbit* o, uint64_t n_cfg, const double* g, const int64_t* cfg_index,
                             double tol_fp, double* lambda1, uint8_t* region, int64_t* n_in_region,
                             int32_t* lanczos_steps, void* cuda_stream) {
    t_launches = 0;
    if (!o) return fail(U1GF_EINVAL, "u1gf_check_fp: NULL orbit");
    if (!n_in_region) return fail(U1GF_EINVAL, "u1gf_check_fp: NULL n_in_region");
    if (!(tol_fp >= 0.0)) return fail(U1GF_EINVAL, "u1gf_check_fp: tol_fp must be >= 0");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    U1GF_CUDA(cudaMemsetAsync(n_in_region, 0, sizeof(int64_t), st));
    if (n_cfg == 0) return U1GF_OK;
    if (!g || !lambda1 || !region) return fail(U1GF_EINVAL, "u1gf_check_fp: NULL array");
    FpParams P{n_cfg, (const double2*)g, tol_fp, lambda1, region, (unsigned long long*)n_in_region, lanczos_steps, cfg_index};
    switch (o->dev.d) {
        case 1: return launch<1>(o, P, st);
        case 2: return launch<2>(o, P, st);
        case 3: return launch<3>(o, P, st);
        default: return launch<4>(o, P, st);
    }
}
