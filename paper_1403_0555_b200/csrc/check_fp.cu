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

// ASYNC kernels carry one extra warp (the last) that runs the Ritz tests: barrier 1 joins the compute warps, barrier 2
// the whole CTA (rendezvous with the Ritz warp); the other kernels use the ordinary CTA barrier.
template <bool ASYNC>
__device__ __forceinline__ void compute_barrier() {
    if (ASYNC) asm volatile("bar.sync 1, %0;" ::"r"(blockDim.x - 32) : "memory");
    else __syncthreads();
}
__device__ __forceinline__ void cta_barrier() { asm volatile("bar.sync 2, %0;" ::"r"(blockDim.x) : "memory"); }
template <bool ASYNC>
__device__ __forceinline__ int compute_warps() { return ASYNC ? (int)((blockDim.x - 32) >> 5) : (int)((blockDim.x + 31) >> 5); }

template <bool ASYNC>
__device__ __forceinline__ double block_sum(double a, double (*red)[32], int& buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = compute_warps<ASYNC>();
    if (lane == 0) red[buf][warp] = a;
    compute_barrier<ASYNC>();
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
template <bool ASYNC>
__device__ __forceinline__ void block_sum2(double& a, double& b, double (*red2)[32][2], int& buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = compute_warps<ASYNC>();
    if (lane == 0) {
        red2[buf][warp][0] = a;
        red2[buf][warp][1] = b;
    }
    compute_barrier<ASYNC>();
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

// History of the Ritz tests of one configuration (registers of the warp that runs them) and one test.
struct RitzState {
    double lam, lam_hi, res_prev, last_drop;
    int k_prev, n_checks;
    bool have_drop;
    __device__ void reset(int dim) {
        lam = 0.0; lam_hi = 4.0 * dim + 1.0; res_prev = 0.0; last_drop = 0.0;
        k_prev = 0; n_checks = 0; have_drop = false;
    }
};

// Test of T_k by one warp (all 32 lanes call this): smallest Ritz value `l`, residual bound `res`, and `step`, the
// distance from k to where the bound, which falls geometrically, is expected to cross 1e-10.  final: refine the Ritz
// value whatever the residual (breakdown or step cap).
template <int DIM>
__device__ void ritz_test(RitzState& R, const double* alpha, const double* beta, const double* beta2, const double* ibeta,
                          int k, bool breakdown, bool final, double& l, double& res, int& step) {
    // Ritz values decrease with k (interlacing): the new one lies below the last; a lower end a few times the last
    // decrease below it is tried first (one Sturm count says whether it holds)
    double lo_try = -(4.0 * DIM + 1.0);
    if (R.have_drop) {
        const double cand = R.lam - 8.0 * R.last_drop - 1e-9;
        if (sturm_count(alpha, beta2, k, cand) == 0) lo_try = cand;
    }
    // the Ritz value to 1e-11 is enough to follow the residual; it is refined to 2e-14 once the test passes
    l = smallest_ritz(alpha, beta2, k, lo_try, R.lam_hi, 1e-11);
    res = breakdown ? 0.0 : beta[k - 1] * last_component(alpha, beta, ibeta, k, l - 1e-13);
    if (final || res < 1e-10) l = smallest_ritz(alpha, beta2, k, l - 2e-11 * fmax(1.0, fabs(l)), l + 2e-11 * fmax(1.0, fabs(l)), 2e-14);
    if (R.n_checks > 0) {
        R.last_drop = fmax(R.lam - l, 0.0);
        R.have_drop = true;
    }
    R.lam = l;
    R.lam_hi = l + 1e-9;
    step = max(4, k / 4);
    if (R.n_checks > 0 && res > 0.0 && res < R.res_prev) {   // (a measured decay may carry the next test up to k/2 ahead)
        const double per_step = log(R.res_prev / res) / (double)(k - R.k_prev);
        step = max(3, min(max(4, k / 2), (int)(0.9 * log(res / 1e-10) / per_step) + 1));
    }
    R.res_prev = res;
    R.k_prev = k;
    ++R.n_checks;
}

// Mailbox between the compute warps and the Ritz warp of an ASYNC kernel (shared memory).  A rendezvous is two CTA
// barriers: before the first the compute side has written the command and the Ritz warp the verdict of its last test;
// between the two each side reads the other's fields into registers; after the second both may write again.
struct RitzMail {
    int cmd_k;       // > 0: test T_k; 0: nothing (the compute side only wants the verdict); < 0: leave
    int cmd_flags;   // 1: first test of a configuration (forget the history); 2: final; 4: breakdown
    int v_k, v_step; // verdict: the k it belongs to; predicted distance to the crossing
    double v_lam, v_res;
};

// One CTA per configuration, every compute thread owns up to SPT sites (i = tid, tid + T, ...).  The neighbour indices
// of a thread's sites are the same for every configuration and every step: they are read once into registers (16-bit,
// V <= 8192) instead of 2 DIM index loads per site and mat-vec.  Per Lanczos step: the mat-vec with <w, v1> (one
// reduction), w -= alpha v1 with the mean of w and its norm without the mean, sum w^2 - V mean^2, in ONE reduction, then
// the scaled vector -- three barriers per step.
// The Ritz test is serial work of one warp.  Small lattices (several CTAs per SM): warp 0 runs it while the others wait;
// other configurations fill the SM.  ASYNC (the large lattices, one or two CTAs per SM, where nothing else fills the
// gap): an extra warp runs the test concurrently with the following Lanczos steps, which only append to the coefficient
// arrays; at a test point the compute warps hand over T_k and pick up the verdict of the PREVIOUS test.  A configuration
// ends at the first test that passes, in test order; which tests are made depends only on the data, never on timing, so
// lambda_1, region and step count are reproducible; the few steps taken after the passing test are discarded.
template <int DIM, int SPT, int MAXT, bool ASYNC>
__global__ void __launch_bounds__(MAXT + (ASYNC ? 32 : 0), MAXT <= 256 ? 2 : 1) lanczos_kernel(const OrbitDev D, const FpParams P) {
    extern __shared__ double sm[];
    const int V = D.V, tid = threadIdx.x, T = blockDim.x - (ASYNC ? 32 : 0);
    double* c = sm;                 // [DIM][V]
    double* va = c + (size_t)V * DIM;  // [V]
    double* vb = va + V;            // [V]
    __shared__ double red[2][32];
    __shared__ double red2[2][32][2];
    __shared__ RitzMail mail;
    const int kcap = min(V - 1, kMaxK);
    double* alpha = vb + V;   // Lanczos coefficients [4][kcap], behind the vectors in dynamic shared memory
    double* beta = alpha + kcap;
    double* beta2 = beta + kcap;
    double* ibeta = beta2 + kcap;
    int buf = 0, buf2 = 0;
    const int kmax = kcap;
    RitzState R;
    R.reset(DIM);

    if (ASYNC && tid >= T) {
        // ------------------------------------------------------------------ the Ritz warp
        for (;;) {
            cta_barrier();
            const int k = mail.cmd_k, flags = mail.cmd_flags;
            cta_barrier();
            if (k < 0) break;
            if (k == 0) continue;
            if (flags & 1) R.reset(DIM);
            double l, res;
            int step;
            ritz_test<DIM>(R, alpha, beta, beta2, ibeta, k, (flags & 4) != 0, (flags & 2) != 0, l, res, step);
            if ((tid & 31) == 0) {
                mail.v_k = k;
                mail.v_step = step;
                mail.v_lam = l;
                mail.v_res = res;
            }
            __syncwarp();
        }
        return;
    }

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
    // ASYNC: hand a command to the Ritz warp and pick up its last verdict
    auto rendezvous = [&](int k, int flags, int& vk, int& vstep, double& vlam, double& vres) {
        if (tid == 0) {
            mail.cmd_k = k;
            mail.cmd_flags = flags;
        }
        cta_barrier();
        vk = mail.v_k;
        vstep = mail.v_step;
        vlam = mail.v_lam;
        vres = mail.v_res;
        cta_barrier();
    };

    for (unsigned long long cfg = blockIdx.x; cfg < P.n_cfg; cfg += gridDim.x) {
        const double2* g = P.g + (P.index ? (unsigned long long)P.index[cfg] : cfg) * (unsigned long long)V;
        compute_barrier<ASYNC>();
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
        s1 = block_sum<ASYNC>(s1, red, buf);
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
        s2 = block_sum<ASYNC>(s2, red, buf);
        const double inv0 = rsqrt(s2);
#pragma unroll
        for (int s = 0; s < SPT; ++s) {
            const int i = tid + s * T;
            if (i < V) va[i] *= inv0;
        }
        compute_barrier<ASYNC>();

        double* v1 = va;  // current Lanczos vector
        double* v0 = vb;  // previous one; overwritten by the new direction
        double beta_prev = 0.0, lam = 0.0;
        int k = 0, next_check = 16, n_handed = 0, k_out = 0;
        bool done = false, unconverged = false;
        if (!ASYNC) R.reset(DIM);
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
            a = block_sum<ASYNC>(a, red, buf);
            // w -= alpha v1; its mean (the constant mode, taken out every step) and its norm without the mean
            double sw = 0.0, sww = 0.0;
#pragma unroll
            for (int s = 0; s < SPT; ++s) {
                w[s] = fma(-a, vi[s], w[s]);
                sw += w[s];
                sww = fma(w[s], w[s], sww);
            }
            block_sum2<ASYNC>(sw, sww, red2, buf2);
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
                const bool final = breakdown || k == kmax;
                if (ASYNC) {
                    int vk, vstep;
                    double vlam, vres;
                    rendezvous(k, (n_handed == 0 ? 1 : 0) | (final ? 2 : 0) | (breakdown ? 4 : 0), vk, vstep, vlam, vres);
                    if (n_handed > 0 && vres < 1e-10) {   // the previous test passed: the steps since are discarded
                        lam = vlam;
                        k_out = vk;
                        done = true;
                    } else if (final) {                   // wait for this last test
                        rendezvous(0, 0, vk, vstep, vlam, vres);
                        lam = vlam;
                        k_out = k;
                        unconverged = !breakdown && !(vres < 1e-10) && k < V - 1;   // k = V-1: the Krylov space is the whole of 1-perp, T_k is exact
                        done = true;
                    } else {
                        const int pred = n_handed > 0 ? vk + vstep : k + max(4, k / 4);
                        next_check = max(k + 3, pred);
                    }
                    ++n_handed;
                } else {
                    __syncthreads();
                    if (tid < 32) {
                        double l, res;
                        int step;
                        ritz_test<DIM>(R, alpha, beta, beta2, ibeta, k, breakdown, final, l, res, step);
                        if (tid == 0) {
                            mail.v_lam = l;
                            mail.v_res = res;
                            mail.v_step = step;
                        }
                    }
                    __syncthreads();
                    lam = mail.v_lam;
                    const double res = mail.v_res;
                    k_out = k;
                    if (final || res < 1e-10) done = true;
                    // k = V-1 (reachable only for V-1 <= 512): the Krylov space is the whole of 1-perp and T_k is exact -- in
                    // exact arithmetic.  Without reorthogonalisation that is a heuristic: a run that ends there is reported
                    // as converged whatever its residual bound.  Dropping the exemption was tried (round 3): 4 of 2048
                    // starts of a hot 2^4 orbit and 4 of 2048 of a 6x6 one then carry bit 2, with lambda_1 within 1e-8 of
                    // the dense eigenvalue all the same -- the bound at k = V-1 is made of a roundoff-level beta and says
                    // little.  Kept; stated in include/u1gf.h and DESIGN.md R16.
                    unconverged = !breakdown && !(res < 1e-10) && k < V - 1;
                    next_check = k + mail.v_step;
                }
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
                compute_barrier<ASYNC>();
            }
        }
        if (tid == 0) {
            P.lambda1[cfg] = lam;
            const uint8_t reg = lam > P.tol_fp ? 1 : (fabs(lam) <= P.tol_fp ? 2 : 0);
            // bit 2: the step cap was reached with the residual bound still above 1e-10 (R16): lambda1 is then only an
            // upper bound of the eigenvalue and the caller should not trust a region of 1 or 2
            P.region[cfg] = (uint8_t)(reg | (unconverged ? 4 : 0));
            if (P.steps) P.steps[cfg] = k_out;
            if (reg) atomicAdd(P.n_in, 1ull);
        }
    }
    if (ASYNC) {   // release the Ritz warp
        int vk, vstep;
        double vlam, vres;
        rendezvous(-1, 0, vk, vstep, vlam, vres);
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
    // the large lattices (8 sites per thread: one or two CTAs per SM) run the Ritz test on a warp of its own
#ifndef U1GF_FP_NO_ASYNC
    const bool async = spt == 8;
#else
    const bool async = false;
#endif
    auto kern = spt == 8 ? (async ? (T <= 192 ? lanczos_kernel<DIM, 8, 192, true>      // 6^4: 144 registers at two CTAs per SM
                                     : T <= 256 ? lanczos_kernel<DIM, 8, 256, true>
                                     : T <= 512 ? lanczos_kernel<DIM, 8, 512, true>    // 8^4
                                                : lanczos_kernel<DIM, 8, 640, true>)
                                  : (T <= 256 ? lanczos_kernel<DIM, 8, 256, false> : lanczos_kernel<DIM, 8, 640, false>))
                         : (spt == 4 ? (T <= 256 ? lanczos_kernel<DIM, 4, 256, false> : lanczos_kernel<DIM, 4, 640, false>)
                                     : lanczos_kernel<DIM, 2, 256, false>);
    const int threads = T + (async ? 32 : 0);
    if (T > 640) return fail(U1GF_EINVAL, "u1gf_check_fp: lattice of %d sites does not fit the resident Lanczos kernel", V);
    if (smem > 48 * 1024) U1GF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    U1GF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem));
    if (per_sm < 1) return fail(U1GF_ECUDA, "u1gf_check_fp: kernel does not fit on an SM");
    unsigned long long grid = (unsigned long long)per_sm * o->sm_count;
    if (grid > P.n_cfg) grid = P.n_cfg;
    kern<<<(unsigned)grid, threads, smem, st>>>(o->dev, P);
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
