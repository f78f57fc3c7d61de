// relax_generic.cu -- generic relaxation kernel: one CTA per start, the gauge field g resident in shared
// memory, threads strided over the sites of each update phase.  Valid for every d in 1..4 and every extent
// >= 2 (odd extents through the level phases of reading R3, extent 2 through its double bonds, R4).  The
// specialised resident kernels of relax_lanes.cu cover the small even lattices faster; this one is the
// production path for 3^4, 6^4, 8^4 and the correctness path for everything.
//
// Steps: a2 start generation, a3 half-sweep site update (Eq. 4-5,
// PAPER.md:L79-99), a4 gauge precision and stop rule (R5), a5 functional (Eq. 3),
// a6 canonical form and signature.
#include "u1gf_internal.h"

namespace u1gf {

namespace {

struct Params {
    uint64_t seed, first_start, n_starts;
    const uint64_t* start_ids;
    double omega, eps;
    int max_sweeps, check_every;
    double* F_norm;
    int32_t* sweeps;
    uint8_t* status;
    double* sig;
    double* g_canon;
    unsigned long long* counter;
    // redo mode (R6 fix-up of the resident kernels): the number of starts comes from device memory and entry idx of the
    // work list is the position pos[idx] in the output arrays (and in start_ids); both NULL otherwise
    const unsigned* n_dev;
    const unsigned long long* pos;
    // ensemble mode (the paper's own mapping, one lattice per block with the grid over the samples of all
    // orbits): work item k is start first_start + k % ens_n_per of orbit k / ens_n_per, whose links are at
    // ens_U + orbit * V * DIM and whose start seed is ens_seeds[orbit]; n_starts = n_orbits * ens_n_per.  NULL otherwise
    const double2* ens_U;
    const unsigned long long* ens_seeds;
    unsigned long long ens_n_per;
};

// w_i = sum_mu [ conj(U_{i,mu}) g_{i+mu} + U_{i-mu,mu} g_{i-mu} ]   (= conj K_i of Eq. 5)
template <int DIM>
__device__ __forceinline__ void neighbour_sum(const OrbitDev& D, const double2* __restrict__ U,
                                              const double2* __restrict__ g, int i, double& wr, double& wi) {
    wr = 0.0;
    wi = 0.0;
#pragma unroll
    for (int mu = 0; mu < DIM; ++mu) {
        const int jf = __ldg(D.fwd + i * DIM + mu);
        const int jb = __ldg(D.bwd + i * DIM + mu);
        const double2 u = __ldg(U + i * DIM + mu);
        const double2 b = __ldg(U + jb * DIM + mu);
        const double2 gf = g[jf];
        const double2 gb = g[jb];
        wr = fma(u.x, gf.x, wr);
        wr = fma(u.y, gf.y, wr);
        wi = fma(u.x, gf.y, wi);
        wi = fma(-u.y, gf.x, wi);
        wr = fma(b.x, gb.x, wr);
        wr = fma(-b.y, gb.y, wr);
        wi = fma(b.x, gb.y, wi);
        wi = fma(b.y, gb.x, wi);
    }
}

// local solution g^ = w/|w| mixed by over-relaxation and re-projected (R2); R6 skip.
__device__ __forceinline__ double2 site_update(double2 gi, double wr, double wi, double omega, bool& skipped) {
    const double n = fma(wr, wr, wi * wi);
    if (n < 1e-280) {
        skipped = true;
        return gi;
    }
    const double c = omega * rsqrt(n);
    const double om1 = 1.0 - omega;
    const double hr = fma(om1, gi.x, c * wr);
    const double hi = fma(om1, gi.y, c * wi);
    const double r2 = rsqrt(fma(hr, hr, hi * hi));
    return make_double2(hr * r2, hi * r2);
}

// Sum of two per-thread values over the CTA, same result in every thread, fixed tree: shuffle-down inside each
// warp, then every thread adds the warp partials in warp order.  `buf` alternates so that one barrier is enough.
__device__ __forceinline__ void block_sum2(double& a, double& b, double (*red)[32][2], int& buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) {
        red[buf][warp][0] = a;
        red[buf][warp][1] = b;
    }
    __syncthreads();
    double sa = 0.0, sb = 0.0;
    for (int w = 0; w < nw; ++w) {
        sa += red[buf][w][0];
        sb += red[buf][w][1];
    }
    a = sa;
    b = sb;
    buf ^= 1;
}

template <int DIM, int MAXS>
__global__ void __launch_bounds__(1024) relax_generic_kernel(const OrbitDev D, const Params P) {
    extern __shared__ double2 g[];  // [V]
    __shared__ double red[2][32][2];
    __shared__ unsigned long long s_next;
    const int tid = threadIdx.x, T = blockDim.x, V = D.V;
    int buf = 0;
    const double invV = 1.0;  // division by V is done explicitly below, as the stop rule is written (R5)
    (void)invV;

    for (;;) {
        if (tid == 0) s_next = atomicAdd(P.counter, 1ull);
        __syncthreads();
        unsigned long long k = s_next;
        if (k >= (P.n_dev ? (unsigned long long)*P.n_dev : P.n_starts)) break;
        if (P.pos) k = P.pos[k];
        uint64_t s = P.start_ids ? P.start_ids[k] : P.first_start + k;
        uint64_t seed = P.seed;
        const double2* __restrict__ U = D.U;
        if (P.ens_U) {   // the orbit this start belongs to (results stay at position k)
            const unsigned long long orb = k / P.ens_n_per;
            s = P.first_start + (k - orb * P.ens_n_per);
            seed = P.ens_seeds[orb];
            U = P.ens_U + orb * (unsigned long long)(V * DIM);
        }

        // a2: random start
        for (int i = tid; i < V; i += T) {
            const u32x4 r = philox((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 0u, (uint32_t)seed,
                                   (uint32_t)(seed >> 32));
            double sn, cs;
            sincospi(unit_interval_pm1(r.x, r.y), &sn, &cs);
            g[i] = make_double2(cs, sn);
        }
        __syncthreads();

        int t = 0;
        bool skipped = false, converged = false;
        double Ftot = 0.0;
        if (D.all_even) {
            // two colours; the gauge precision of the field after sweep t comes for free: odd sites from the w
            // just used (their neighbours do not move any more), even sites from the w formed at the start of
            // sweep t+1, deciding before anything is written (R5).
            const int off0 = D.phase_off[0], off1 = D.phase_off[1], off2 = D.phase_off[2];
            double accO = 0.0;
            for (;;) {
                double accE = 0.0, Fp = 0.0;
                double2 gnew[MAXS];
                int site[MAXS];
#pragma unroll
                for (int j = 0; j < MAXS; ++j) {
                    const int q = off0 + tid + j * T;
                    site[j] = -1;
                    if (q < off1) {
                        const int i = __ldg(D.order + q);
                        site[j] = i;
                        double wr, wi;
                        neighbour_sum<DIM>(D, U, g, i, wr, wi);
                        const double2 gi = g[i];
                        const double dl = fma(gi.y, wr, -gi.x * wi);  // Delta_i = Im(g_i conj w_i)
                        accE = fma(dl, dl, accE);
                        Fp += fma(gi.x, wr, gi.y * wi);  // Re(g_i conj w_i): every link has one even end
                        gnew[j] = site_update(gi, wr, wi, P.omega, skipped);
                    }
                }
                double S = accE + accO;
                block_sum2(S, Fp, red, buf);
                Ftot = Fp;
                if (t > 0 && t % P.check_every == 0 && S / (double)V < P.eps) {
                    converged = true;
                    break;
                }
                if (t == P.max_sweeps) break;
#pragma unroll
                for (int j = 0; j < MAXS; ++j)
                    if (site[j] >= 0) g[site[j]] = gnew[j];
                __syncthreads();
                accO = 0.0;
#pragma unroll
                for (int j = 0; j < MAXS; ++j) {
                    const int q = off1 + tid + j * T;
                    if (q < off2) {
                        const int i = __ldg(D.order + q);
                        double wr, wi;
                        neighbour_sum<DIM>(D, U, g, i, wr, wi);
                        const double2 gn = site_update(g[i], wr, wi, P.omega, skipped);
                        g[i] = gn;
                        const double dl = fma(gn.y, wr, -gn.x * wi);
                        accO = fma(dl, dl, accO);
                    }
                }
                __syncthreads();
                ++t;
            }
        } else {
            // odd extents (R3): level phases, then a separate residual pass (a same-parity neighbour may still
            // move after w_i was formed, so the fused measure above is not exact here).
            for (;;) {
                for (int p = 0; p < D.n_phases; ++p) {
                    for (int q = D.phase_off[p] + tid; q < D.phase_off[p + 1]; q += T) {
                        const int i = __ldg(D.order + q);
                        double wr, wi;
                        neighbour_sum<DIM>(D, U, g, i, wr, wi);
                        g[i] = site_update(g[i], wr, wi, P.omega, skipped);
                    }
                    __syncthreads();
                }
                ++t;
                const bool check = t % P.check_every == 0;
                if (check || t == P.max_sweeps) {
                    double S = 0.0, Fp = 0.0;
                    for (int i = tid; i < V; i += T) {
                        double wr, wi;
                        neighbour_sum<DIM>(D, U, g, i, wr, wi);
                        const double2 gi = g[i];
                        const double dl = fma(gi.y, wr, -gi.x * wi);
                        S = fma(dl, dl, S);
                        Fp += 0.5 * fma(gi.x, wr, gi.y * wi);  // each link is seen from both ends
                    }
                    block_sum2(S, Fp, red, buf);
                    Ftot = Fp;
                    if (check && S / (double)V < P.eps) {
                        converged = true;
                        break;
                    }
                    if (t == P.max_sweeps) break;
                }
            }
        }
        const int any_skip = __syncthreads_or(skipped ? 1 : 0);

        // a6: canonical form g~ = g conj(g_{V-1}) and signature
        const double2 c = g[V - 1];
        double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
        for (int i = tid; i < V; i += T) {
            const double2 gi = g[i];
            const double re = fma(gi.x, c.x, gi.y * c.y);
            const double im = fma(gi.y, c.x, -gi.x * c.y);
            const unsigned bits = __ldg(D.sgn + i);
            p0 += ((bits & 1u) ? re : -re) + ((bits & 16u) ? im : -im);
            p1 += ((bits & 2u) ? re : -re) + ((bits & 32u) ? im : -im);
            p2 += ((bits & 4u) ? re : -re) + ((bits & 64u) ? im : -im);
            p3 += ((bits & 8u) ? re : -re) + ((bits & 128u) ? im : -im);
            if (P.g_canon) reinterpret_cast<double2*>(P.g_canon)[k * (unsigned long long)V + i] = make_double2(re, im);
        }
        block_sum2(p0, p1, red, buf);
        block_sum2(p2, p3, red, buf);
        if (tid == 0) {
            P.F_norm[k] = Ftot / ((double)DIM * (double)V);
            P.sweeps[k] = t;
            P.status[k] = (uint8_t)((converged ? 0 : 1) | (any_skip ? 2 : 0));
            double4 sg = make_double4(p0 / (double)V, p1 / (double)V, p2 / (double)V, p3 / (double)V);
            reinterpret_cast<double4*>(P.sig)[k] = sg;
        }
        // the barrier after the next atomicAdd separates these reads of g from the next start's writes
    }
}

struct Launch {
    int T, maxs;
};

Launch pick(const u1gf_orbit* o) {
    const int mp = o->dev.max_phase;
    for (int k : {1, 2, 4}) {
        const int T = ((mp + k - 1) / k + 31) / 32 * 32;
        if (T <= 1024) return {T < 32 ? 32 : T, k};
    }
    return {1024, 4};
}

template <int DIM, int MAXS>
int launch(const u1gf_orbit* o, const Params& P, int T, cudaStream_t st, bool redo = false) {
    auto kern = relax_generic_kernel<DIM, MAXS>;
    const size_t smem = (size_t)o->dev.V * sizeof(double2);
    if (smem > 48 * 1024) U1GF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    U1GF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T, smem));
    if (per_sm < 1) return fail(U1GF_ECUDA, "generic relaxation kernel does not fit on an SM (V = %d)", o->dev.V);
    unsigned long long grid = (unsigned long long)per_sm * (unsigned long long)o->sm_count;
    if (grid > P.n_starts) grid = P.n_starts;
    if (redo) {   // the caller zeroed the counter
        kern<<<(unsigned)grid, T, smem, st>>>(o->dev, P);
        U1GF_CUDA(cudaGetLastError());
        ++t_launches;
        return U1GF_OK;
    }
    U1GF_CUDA(cudaMemsetAsync(P.counter, 0, sizeof(unsigned long long), st));
    kern<<<(unsigned)grid, T, smem, st>>>(o->dev, P);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    return U1GF_OK;
}

template <int DIM>
int launch_d(const u1gf_orbit* o, const Params& P, Launch L, cudaStream_t st, bool redo = false) {
    switch (L.maxs) {
        case 1: return launch<DIM, 1>(o, P, L.T, st, redo);
        case 2: return launch<DIM, 2>(o, P, L.T, st, redo);
        default: return launch<DIM, 4>(o, P, L.T, st, redo);
    }
}

}  // namespace

size_t generic_workspace_bytes(const u1gf_orbit*, uint64_t) { return 256; }

int generic_relax_list(const u1gf_orbit* o, const RelaxArgs& a, const unsigned* n_dev, const unsigned long long* pos,
                       unsigned long long* counter, cudaStream_t st) {
    Params P{a.seed, a.first_start, a.n_starts, a.start_ids, a.omega, a.eps, a.max_sweeps, a.check_every,
             a.F_norm, a.sweeps, a.status, a.sig, a.g_canon, counter, n_dev, pos, nullptr, nullptr, 0ull};
    // a small grid: the list is empty unless a neighbour sum vanished somewhere (R6)
    if (P.n_starts > 4ull * (unsigned long long)o->sm_count) P.n_starts = 4ull * (unsigned long long)o->sm_count;
    const Launch L = pick(o);
    switch (o->dev.d) {
        case 1: return launch_d<1>(o, P, L, st, true);
        case 2: return launch_d<2>(o, P, L, st, true);
        case 3: return launch_d<3>(o, P, L, st, true);
        default: return launch_d<4>(o, P, L, st, true);
    }
}

int generic_relax(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st) {
    Params P{a.seed, a.first_start, a.n_starts, a.start_ids, a.omega, a.eps, a.max_sweeps, a.check_every,
             a.F_norm, a.sweeps, a.status, a.sig, a.g_canon, (unsigned long long*)a.workspace, nullptr, nullptr,
             nullptr, nullptr, 0ull};
    const Launch L = pick(o);
    switch (o->dev.d) {
        case 1: return launch_d<1>(o, P, L, st);
        case 2: return launch_d<2>(o, P, L, st);
        case 3: return launch_d<3>(o, P, L, st);
        default: return launch_d<4>(o, P, L, st);
    }
}

// Ensemble mode: a.n_starts starts of each of n_orbits orbits of the shape of `o` in one launch (a.seed is not used).
int generic_relax_ens(const u1gf_orbit* o, const double2* U_all, const unsigned long long* seeds, unsigned n_orbits,
                      const RelaxArgs& a, cudaStream_t st) {
    Params P{0, a.first_start, a.n_starts * (uint64_t)n_orbits, nullptr, a.omega, a.eps, a.max_sweeps, a.check_every,
             a.F_norm, a.sweeps, a.status, a.sig, nullptr, (unsigned long long*)a.workspace, nullptr, nullptr,
             U_all, seeds, (unsigned long long)a.n_starts};
    const Launch L = pick(o);
    switch (o->dev.d) {
        case 1: return launch_d<1>(o, P, L, st);
        case 2: return launch_d<2>(o, P, L, st);
        case 3: return launch_d<3>(o, P, L, st);
        default: return launch_d<4>(o, P, L, st);
    }
}

}  // namespace u1gf
