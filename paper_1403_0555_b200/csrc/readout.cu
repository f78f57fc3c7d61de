// readout.cu -- SURVEY section 8(f)-3, the part after the launch: what the paper reads off an ensemble of orbits.
//   * u1gf_ensemble_stats: per orbit the value of the functional at the best copy found, x_g = 1 - max F/(dV) (the paper's
//     "global minimum", Tab. III), and over the orbits the average and standard deviation of the number
//     of copies (Tab. I), of x_g (Tab. III) and of the number of copies inside the first Gribov region (L9, L50).
//   * u1gf_relative_deviation_hist: the distribution of (x_i - x_g)/x_g over the samples of an orbit, averaged over the
//     orbits (Fig. 8).
//   * u1gf_hist_ratio: bin by bin, the ratio of the entries of two histograms of the same orbits taken with different
//     numbers of samples, and the bins only the larger run fills (Fig. 5).
// Inputs are the arrays u1gf_relax_ensemble / u1gf_count_copies_ensemble leave on the device.  Integer work is done with
// integer atomics; every floating-point sum runs in a fixed order (one thread, orbit after orbit), and where a floating-
// point value decides a bin the operations are single IEEE operations without contraction, so the integer outputs do not
// depend on the launch configuration.
#include "u1gf_internal.h"

namespace u1gf {
namespace {

// one CTA per orbit: x_g = 1 - max over the copies of F/(dV) at the leader
__global__ void __launch_bounds__(256) best_x_kernel(unsigned long long n_per, const double* __restrict__ F,
                                                     const long long* __restrict__ rep, const long long* __restrict__ n_distinct,
                                                     double* __restrict__ best_x) {
    __shared__ double red[256];
    const unsigned long long o = blockIdx.x, base = o * n_per;
    const long long nd = n_distinct[o];
    double m = -INFINITY;
    for (long long c = threadIdx.x; c < nd; c += blockDim.x) m = fmax(m, F[base + (unsigned long long)rep[base + c]]);
    red[threadIdx.x] = m;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) red[threadIdx.x] = fmax(red[threadIdx.x], red[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) best_x[o] = nd > 0 ? __dsub_rn(1.0, red[0]) : nan("");
}

// mean and sample standard deviation (n - 1 in the denominator, 0 for a single value) of v_0 .. v_{n-1}, in index order
template <class Get>
__device__ void mean_std(int n, Get get, double& mean, double& sd) {
    double s = 0.0;
    int m = 0;
    for (int o = 0; o < n; ++o) {
        const double v = get(o);
        if (v == v) {
            s = __dadd_rn(s, v);
            ++m;
        }
    }
    mean = m ? __ddiv_rn(s, (double)m) : nan("");
    double q = 0.0;
    for (int o = 0; o < n; ++o) {
        const double v = get(o);
        if (v == v) {
            const double e = __dsub_rn(v, mean);
            q = __dadd_rn(q, __dmul_rn(e, e));
        }
    }
    sd = m > 1 ? sqrt(__ddiv_rn(q, (double)(m - 1))) : (m == 1 ? 0.0 : nan(""));
}

__global__ void stats_kernel(int n_orbits, const long long* __restrict__ n_distinct, const long long* __restrict__ n_in_region,
                             const double* __restrict__ best_x, double* __restrict__ stats) {
    if (blockIdx.x || threadIdx.x) return;
    mean_std(n_orbits, [&](int o) { return (double)n_distinct[o]; }, stats[0], stats[1]);
    mean_std(n_orbits, [&](int o) { return best_x[o]; }, stats[2], stats[3]);   // NaN entries (no converged start) are left out
    if (n_in_region) {
        mean_std(n_orbits, [&](int o) { return (double)n_in_region[o]; }, stats[4], stats[5]);
    } else {
        stats[4] = stats[5] = nan("");
    }
    int used = 0;
    for (int o = 0; o < n_orbits; ++o) used += best_x[o] == best_x[o] ? 1 : 0;
    stats[6] = (double)used;
    stats[7] = (double)n_orbits;
}

// one thread per (orbit, copy slot): the samples of the copy go to the bin of its relative deviation
__global__ void reldev_bin_kernel(unsigned long long n_total, unsigned long long n_per, const double* __restrict__ F,
                                  const long long* __restrict__ rep, const long long* __restrict__ mult,
                                  const long long* __restrict__ n_distinct, const double* __restrict__ best_x, double width,
                                  int nbins, unsigned long long* __restrict__ counts, unsigned long long* __restrict__ n_conv) {
    for (unsigned long long p = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; p < n_total;
         p += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long o = p / n_per, c = p - o * n_per;
        if ((long long)c >= n_distinct[o]) continue;
        const double xg = best_x[o];
        if (!(xg > 0.0)) continue;   // no converged start, or the trivial orbit (x_g = 0): no relative deviation
        const double x = __dsub_rn(1.0, F[o * n_per + (unsigned long long)rep[p]]);
        const double dev = __ddiv_rn(__dsub_rn(x, xg), xg);
        const double q = floor(__ddiv_rn(dev, width));
        const int b = q < 0.0 ? 0 : (q >= (double)nbins ? nbins - 1 : (int)q);
        const unsigned long long m = (unsigned long long)mult[p];
        atomicAdd(&counts[o * (unsigned long long)nbins + b], m);
        atomicAdd(&n_conv[o], m);
    }
}

// one thread per bin: the orbit-averaged fraction of samples, summed orbit after orbit
__global__ void reldev_avg_kernel(int n_orbits, int nbins, const unsigned long long* __restrict__ counts,
                                  const unsigned long long* __restrict__ n_conv, double* __restrict__ avg,
                                  long long* __restrict__ n_used) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nbins) return;
    double s = 0.0;
    int used = 0;
    for (int o = 0; o < n_orbits; ++o) {
        const unsigned long long nc = n_conv[o];
        if (nc == 0ull) continue;
        s = __dadd_rn(s, __ddiv_rn((double)counts[(size_t)o * nbins + b], (double)nc));
        ++used;
    }
    avg[b] = used ? __ddiv_rn(s, (double)used) : 0.0;
    if (b == 0) *n_used = used;
}

__global__ void hist_ratio_kernel(int nbins, const long long* __restrict__ small, const long long* __restrict__ big,
                                  double* __restrict__ ratio, unsigned long long* __restrict__ n_only) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    int only_big = 0, only_small = 0;
    if (b < nbins) {
        const long long s = small[b], g = big[b];
        ratio[b] = s > 0 ? __ddiv_rn((double)g, (double)s) : (g > 0 ? INFINITY : nan(""));
        only_big = s == 0 && g > 0;
        only_small = g == 0 && s > 0;
    }
    const unsigned mb = __ballot_sync(0xffffffffu, only_big), ms = __ballot_sync(0xffffffffu, only_small);
    if ((threadIdx.x & 31) == 0) {
        if (mb) atomicAdd(&n_only[0], (unsigned long long)__popc(mb));
        if (ms) atomicAdd(&n_only[1], (unsigned long long)__popc(ms));
    }
}

}  // namespace
}  // namespace u1gf

using namespace u1gf;

extern "C" {

int u1gf_ensemble_stats(int32_t n_orbits, uint64_t n_per_orbit, const double* F_norm, const int64_t* rep,
                        const int64_t* n_distinct, const int64_t* n_in_region, double* best_x, double* stats,
                        void* cuda_stream) {
    t_launches = 0;
    if (n_orbits < 1 || n_per_orbit < 1) return fail(U1GF_EINVAL, "u1gf_ensemble_stats: n_orbits and n_per_orbit must be >= 1");
    if (!F_norm || !rep || !n_distinct || !best_x || !stats) return fail(U1GF_EINVAL, "u1gf_ensemble_stats: NULL array");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    best_x_kernel<<<(unsigned)n_orbits, 256, 0, st>>>((unsigned long long)n_per_orbit, F_norm, (const long long*)rep,
                                                      (const long long*)n_distinct, best_x);
    U1GF_CUDA(cudaGetLastError());
    stats_kernel<<<1, 32, 0, st>>>(n_orbits, (const long long*)n_distinct, (const long long*)n_in_region, best_x, stats);
    U1GF_CUDA(cudaGetLastError());
    t_launches = 2;
    return U1GF_OK;
}

int u1gf_relative_deviation_hist(int32_t n_orbits, uint64_t n_per_orbit, const double* F_norm, const int64_t* rep,
                                 const int64_t* multiplicity, const int64_t* n_distinct, const double* best_x, double dev_max,
                                 int32_t nbins, int64_t* counts, int64_t* n_converged, double* avg, int64_t* n_orbits_used,
                                 void* cuda_stream) {
    t_launches = 0;
    if (n_orbits < 1 || n_per_orbit < 1 || nbins < 1)
        return fail(U1GF_EINVAL, "u1gf_relative_deviation_hist: n_orbits, n_per_orbit and nbins must be >= 1");
    if (!(dev_max > 0.0)) return fail(U1GF_EINVAL, "u1gf_relative_deviation_hist: dev_max must be > 0");
    if (!F_norm || !rep || !multiplicity || !n_distinct || !best_x || !counts || !n_converged || !avg || !n_orbits_used)
        return fail(U1GF_EINVAL, "u1gf_relative_deviation_hist: NULL array");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned long long n_total = (unsigned long long)n_orbits * n_per_orbit;
    U1GF_CUDA(cudaMemsetAsync(counts, 0, (size_t)n_orbits * (size_t)nbins * sizeof(int64_t), st));
    U1GF_CUDA(cudaMemsetAsync(n_converged, 0, (size_t)n_orbits * sizeof(int64_t), st));
    const double width = dev_max / (double)nbins;
    const unsigned long long want = (n_total + 255) / 256;
    const unsigned blocks = (unsigned)(want < 148ull * 16 ? want : 148ull * 16);
    reldev_bin_kernel<<<blocks, 256, 0, st>>>(n_total, (unsigned long long)n_per_orbit, F_norm, (const long long*)rep,
                                              (const long long*)multiplicity, (const long long*)n_distinct, best_x, width, nbins,
                                              (unsigned long long*)counts, (unsigned long long*)n_converged);
    U1GF_CUDA(cudaGetLastError());
    reldev_avg_kernel<<<(unsigned)((nbins + 127) / 128), 128, 0, st>>>(n_orbits, nbins, (const unsigned long long*)counts,
                                                                      (const unsigned long long*)n_converged, avg,
                                                                      (long long*)n_orbits_used);
    U1GF_CUDA(cudaGetLastError());
    t_launches = 2;
    return U1GF_OK;
}

int u1gf_hist_ratio(int32_t nbins, const int64_t* hist_small, const int64_t* hist_big, double* ratio, int64_t* n_only,
                    void* cuda_stream) {
    t_launches = 0;
    if (nbins < 1) return fail(U1GF_EINVAL, "u1gf_hist_ratio: nbins must be >= 1");
    if (!hist_small || !hist_big || !ratio || !n_only) return fail(U1GF_EINVAL, "u1gf_hist_ratio: NULL array");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    U1GF_CUDA(cudaMemsetAsync(n_only, 0, 2 * sizeof(int64_t), st));
    hist_ratio_kernel<<<(unsigned)((nbins + 255) / 256), 256, 0, st>>>(nbins, (const long long*)hist_small, (const long long*)hist_big,
                                                                      ratio, (unsigned long long*)n_only);
    U1GF_CUDA(cudaGetLastError());
    t_launches = 1;
    return U1GF_OK;
}

}  // extern "C"
