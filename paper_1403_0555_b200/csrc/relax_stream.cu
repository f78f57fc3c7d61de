// relax_stream.cu -- streamed "lane per start" relaxation kernel for the large even lattices (6^4, 8^4, ...).
//
// The resident kernels of relax_lanes.cu keep the gauge field of 32 starts in the registers of a team of warps; at
// V = 1296 or 4096 sites that no longer fits on chip (32 starts x 64 KiB = 2 MiB).  Here the field of a team lives in
// HBM / L2 in the layout [site][32 starts] (one 512-byte row per site, the start index fastest), and every half-sweep
// streams the rows of the other parity through the SM:
//   * lane l of every warp of the CTA works on start l of the team, so a neighbour is ONE coalesced 128-bit load of
//     512 contiguous bytes per warp, and a link is one warp-uniform load shared by the 32 starts (the generic kernel
//     pays 2d x 16 bytes of link traffic per site update, this one 2d x 16 / 32);
//   * the warps of the CTA split the sites of the current parity; the CTA barrier between the half-sweeps is the
//     only synchronisation (a team never leaves its SM, so its rows stay coherent through L1);
//   * lane-level refill as in relax_lanes.cu: a start that stops is finalised (a5, a6) and replaced at once by the
//     next start, both done by all threads of the CTA on that start's column of the team buffer.
// Arithmetic of a site update and the stop rule (R5) are those of relax_lanes.cu / the oracle: sweep = even half-sweep,
// odd half-sweep; odd-site Delta from the w just used, even-site Delta from the w formed at the start of the next
// sweep; the even rows are double buffered (A[0], A[1]) so that the pre-update values survive the decision.
#include "u1gf_internal.h"

namespace u1gf {
namespace {

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;

struct StreamParams {
    uint64_t seed, first_start, n_starts;
    const uint64_t* start_ids;
    double k2, eps;   // k2 = omega / (1 - omega) (unused when omega == 1)
    int max_sweeps, check_every;
    double* F_norm;
    int32_t* sweeps;
    uint8_t* status;
    double* sig;
    double* g_canon;
    double2* team_buf;             // [teams][2][V][32]
    unsigned long long* counter;   // next start position to hand out
    OrbitDev D;
};

// sum over the CTA of NV per-thread values, same result in every thread, fixed order (deterministic)
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double (*red)[kWarps][NV], int& buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int q = 0; q < NV; ++q) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0)
#pragma unroll
        for (int q = 0; q < NV; ++q) red[buf][warp][q] = v[q];
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NV; ++q) {
        double s = 0.0;
        for (int w = 0; w < kWarps; ++w) s += red[buf][w][q];
        v[q] = s;
    }
    buf ^= 1;
}

__device__ __noinline__ bool r6_vanishes(double nw) {
    return (unsigned long long)__double_as_longlong(nw) < (unsigned long long)__double_as_longlong(1e-280);
}

// a3 for one site of one start: g <- normalise((1-omega) g + omega w/|w|) (R2) in the 8d+20 form of
// relax_lanes.cu (h' = g + (k2/|w|) w = h/(1-omega), second-order rsqrt polish); W1: omega == 1, g <- w/|w|.
template <bool W1>
__device__ __forceinline__ double2 site_update(double2 g, double wr, double wi, double k2, bool& skipped) {
    const double nw = fma(wr, wr, wi * wi);
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(nw));
    const double e = fma(nw * y, -y, 1.0);
    double2 gn;
    if (W1) {
        const double rs = fma(fma(e, 0.375, 0.5), y * e, y);
        gn = make_double2(wr * rs, wi * rs);
    } else {
        const double c = fma(y * (0.5 * k2), e, y * k2);
        const double hr = fma(c, wr, g.x), hi = fma(c, wi, g.y);
        const double nh = fma(hr, hr, hi * hi);
        double y2;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y2) : "d"(nh));
        const double e2 = fma(nh * y2, -y2, 1.0);
        const double r2 = fma(y2 * -0.5, e2, -y2);
        gn = make_double2(hr * r2, hi * r2);
    }
    if (__double2hiint(nw) <= __double2hiint(1e-280)) {   // R6
        if (r6_vanishes(nw)) {
            gn = g;
            skipped = true;
        }
    }
    return gn;
}

template <int DIM>
__device__ __forceinline__ int parity_of(const OrbitDev& D, int i) {
    int p = 0;
#pragma unroll
    for (int mu = 0; mu < DIM; ++mu) {   // unrolled: constant indices keep the orbit descriptor in the constant bank
        p += i % D.ext[mu];
        i /= D.ext[mu];
    }
    return p & 1;
}

// How a half-sweep finds its sites.  Tables: the orbit's order / fwd / bwd arrays, site by site (any all-even lattice;
// three dependent global loads before the first row can be requested).  Cubic<N>: N^DIM lattices with N a compile-time
// constant are walked block-wise by half_sweep_blocks() with pure integer arithmetic.
template <int DIM>
struct Tables {
    static constexpr int kBlocksN = 0;   // no block-wise half-sweep
    __device__ static __forceinline__ void locate(const OrbitDev& D, int p, int r, int& i, int (&jf)[DIM], int (&jb)[DIM]) {
        i = __ldg(D.order + p * D.phase_off[1] + r);
#pragma unroll
        for (int mu = 0; mu < DIM; ++mu) {
            jf[mu] = __ldg(D.fwd + i * DIM + mu);
            jb[mu] = __ldg(D.bwd + i * DIM + mu);
        }
    }
};

template <int DIM, int N>
struct Cubic {
    static_assert(N % 2 == 0, "even extent");
    static constexpr int kBlocksN = N;   // extent for the block-wise half-sweep
};

// w_i = sum_mu [ conj(U_{i,mu}) g_{i+mu} + U_{i-mu,mu} g_{i-mu} ]   (= conj K_i of Eq. 5) for the start of
// this lane; `nb` = rows of the other parity.  Link loads are warp-uniform (one sector each).
template <int DIM>
__device__ __forceinline__ void neighbour_sum(const OrbitDev& D, const double2* __restrict__ nb, int i, const int (&jf)[DIM],
                                              const int (&jb)[DIM], int lane, double& wr, double& wi) {
    // all 2d links and 2d rows in flight before the first FMA (ncu: with the link loads left inside the FMA loop,
    // 46 % of the warp time sat on the long scoreboard of the second FMA -- the links miss L1, the rows evict them)
    double2 gf[DIM], gb[DIM], uf[DIM], ub[DIM];
#pragma unroll
    for (int mu = 0; mu < DIM; ++mu) {
        uf[mu] = __ldg(D.U + i * DIM + mu);
        ub[mu] = __ldg(D.U + jb[mu] * DIM + mu);
    }
#pragma unroll
    for (int mu = 0; mu < DIM; ++mu) {
        gf[mu] = nb[(size_t)jf[mu] * 32 + lane];
        gb[mu] = nb[(size_t)jb[mu] * 32 + lane];
    }
    wr = 0.0;
    wi = 0.0;
#pragma unroll
    for (int mu = 0; mu < DIM; ++mu) {
        wr = fma(uf[mu].x, gf[mu].x, wr);
        wi = fma(uf[mu].x, gf[mu].y, wi);
        wr = fma(uf[mu].y, gf[mu].y, wr);
        wi = fma(-uf[mu].y, gf[mu].x, wi);
        wr = fma(ub[mu].x, gb[mu].x, wr);
        wi = fma(ub[mu].x, gb[mu].y, wi);
        wr = fma(-ub[mu].y, gb[mu].y, wr);
        wi = fma(ub[mu].y, gb[mu].x, wi);
    }
}

// Half-sweep of parity PAR over the 2^DIM blocks of an N^DIM lattice that warp `warp` owns (blocks warp, warp+16, ...).
// The 2^(DIM-1) sites of the other parity inside a block are loaded once into registers and serve DIM of the 2 DIM
// neighbours of each of the block's sites (as in the resident kernels); the other DIM neighbours, the site itself and
// the links come from L1 / L2.  Per site: DIM + 1 + 1/.. row loads instead of 2 DIM + 1.
//   src / dst  rows holding the parity-PAR sites before / after the update (the same array for the odd half-sweep)
//   oth        rows of the other parity
// Returns sum Delta_i^2 of this warp's sites for the lane's start: PAR == 0 measured before the update, 1 after it.
template <int DIM, int N, int PAR, bool W1>
__device__ __forceinline__ double half_sweep_blocks(const OrbitDev& D, const double2* src, double2* dst, const double2* oth,
                                                    int warp, int lane, double k2, bool commit, bool& skipped) {
    constexpr int NB1 = N / 2, HB = 1 << (DIM - 1);
    int nblk = 1;
#pragma unroll
    for (int mu = 0; mu < DIM; ++mu) nblk *= NB1;
    double acc = 0.0;
    for (int b = warp; b < nblk; b += kWarps) {
        int o[DIM], base = 0, rest = b, stride = 1;
#pragma unroll
        for (int mu = 0; mu < DIM; ++mu) {
            o[mu] = 2 * (rest % NB1);
            rest /= NB1;
            base += o[mu] * stride;
            stride *= N;
        }
        // local site l (one bit per direction) sits at base + off(l); parity of l = popc(l) (block origins are even)
        auto off = [](int l) {
            int r = 0, st = 1;
#pragma unroll
            for (int mu = 0; mu < DIM; ++mu) {
                r += ((l >> mu) & 1) * st;
                st *= N;
            }
            return r;
        };
        double2 in[HB];   // the block's sites of the other parity, by half index l >> 1
#pragma unroll
        for (int h = 0; h < HB; ++h) {
            const int l = 2 * h + (((__popc(h) & 1) != (1 - PAR)) ? 1 : 0);
            in[h] = oth[(size_t)(base + off(l)) * 32 + lane];
        }
#pragma unroll
        for (int h = 0; h < HB; ++h) {
            const int l = 2 * h + (((__popc(h) & 1) != PAR) ? 1 : 0);
            const int i = base + off(l);
            const double2 g = __ldcs(src + (size_t)i * 32 + lane);
            double2 gf[DIM], gb[DIM], uf[DIM], ub[DIM];
            int st = 1;
#pragma unroll
            for (int mu = 0; mu < DIM; ++mu) {
                const int ln = l ^ (1 << mu);   // the in-block neighbour along mu
                if (((l >> mu) & 1) == 0) {     // forward neighbour inside, backward one outside (periodic)
                    const int jb = (o[mu] == 0) ? i + (N - 1) * st : i - st;
                    gf[mu] = in[ln >> 1];
                    gb[mu] = oth[(size_t)jb * 32 + lane];
                    ub[mu] = __ldg(D.U + jb * DIM + mu);
                } else {                        // backward neighbour inside, forward one outside (periodic)
                    const int jf = (o[mu] + 2 == N) ? i + st - N * st : i + st;
                    gf[mu] = oth[(size_t)jf * 32 + lane];
                    gb[mu] = in[ln >> 1];
                    ub[mu] = __ldg(D.U + (i - st) * DIM + mu);
                }
                uf[mu] = __ldg(D.U + i * DIM + mu);
                st *= N;
            }
            double wr = 0.0, wi = 0.0;
#pragma unroll
            for (int mu = 0; mu < DIM; ++mu) {   // w_i (= conj K_i of Eq. 5)
                wr = fma(uf[mu].x, gf[mu].x, wr);
                wi = fma(uf[mu].x, gf[mu].y, wi);
                wr = fma(uf[mu].y, gf[mu].y, wr);
                wi = fma(-uf[mu].y, gf[mu].x, wi);
                wr = fma(ub[mu].x, gb[mu].x, wr);
                wi = fma(ub[mu].x, gb[mu].y, wi);
                wr = fma(-ub[mu].y, gb[mu].y, wr);
                wi = fma(ub[mu].y, gb[mu].x, wi);
            }
            if (PAR == 0) {
                const double dl = fma(g.y, wr, -g.x * wi);   // Delta_i of the field after sweep t
                acc = fma(dl, dl, acc);
            }
            bool sk = false;
            const double2 gn = site_update<W1>(g, wr, wi, k2, sk);
            if (commit) {
                __stcs(dst + (size_t)i * 32 + lane, gn);
                if (PAR == 1) {
                    const double dl = fma(gn.y, wr, -gn.x * wi);   // Delta_i = Im(g_i conj w_i) after the update
                    acc = fma(dl, dl, acc);
                }
                skipped |= sk;
            }
        }
    }
    return acc;
}

template <int DIM, bool W1, class IDX>
__global__ void __launch_bounds__(kThreads, 1) relax_stream_kernel(const StreamParams P) {
    constexpr unsigned FULL = 0xffffffffu;
    __shared__ double red[2][kWarps][5];
    __shared__ double sred[2][kWarps][32];
    __shared__ unsigned long long s_pos[32];
    __shared__ unsigned s_skip[32];
    __shared__ unsigned long long s_k;
    const OrbitDev& D = P.D;
    const int V = D.V, half = D.phase_off[1];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double2* const A0 = P.team_buf + (size_t)blockIdx.x * 2 * V * 32;
    double2* const A1 = A0 + (size_t)V * 32;
    auto rows = [&](int buf) { return buf ? A1 : A0; };

    bool active = false, fresh = false, maxed = false, skipped = false;
    int t = 0, eb = 0, rb = 0, fb = 0;
    double accO = 0.0;
    unsigned need = FULL, dumpm = 0;   // first pass: every lane needs a start, nothing to finalise

    for (;;) {
        // ---------------------------------------------------------- service (CTA-uniform): finalise, refill
        for (unsigned m = need; m; m &= m - 1) {
            const int L = __ffs(m) - 1;
            if ((dumpm >> L) & 1u) {
                // a5, a6 for the start of lane L: even rows before the last even half-sweep (A[eb]), odd rows A0
                if (skipped) atomicOr(&s_skip[lane], 1u);
                const int tL = __shfl_sync(FULL, t, L);
                const int mxL = __shfl_sync(FULL, maxed ? 1 : 0, L);
                const unsigned long long k = s_pos[L];
                const double2* E = rows(eb);
                const int pc = parity_of<DIM>(D, V - 1);
                const double2 c = (pc ? A0 : E)[(size_t)(V - 1) * 32 + L];
                double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
                for (int i = tid; i < V; i += kThreads) {
                    const int pi = parity_of<DIM>(D, i);
                    const double2 gi = (pi ? A0 : E)[(size_t)i * 32 + L];
                    const double2* N = pi ? E : A0;   // neighbours have the other parity
#pragma unroll
                    for (int mu = 0; mu < DIM; ++mu) {   // F = sum Re(g_i U_{i,mu} conj g_{i+mu})   (Eq. 3)
                        const double2 u = __ldg(D.U + i * DIM + mu);
                        const double2 gj = N[(size_t)__ldg(D.fwd + i * DIM + mu) * 32 + L];
                        const double ar = fma(gi.x, u.x, -gi.y * u.y), ai = fma(gi.x, u.y, gi.y * u.x);
                        v[0] += fma(ar, gj.x, ai * gj.y);
                    }
                    const double re = fma(gi.x, c.x, gi.y * c.y);   // g~ = g conj(g_{V-1})
                    const double im = fma(gi.y, c.x, -gi.x * c.y);
                    const unsigned bits = __ldg(D.sgn + i);
                    v[1] += ((bits & 1u) ? re : -re) + ((bits & 16u) ? im : -im);
                    v[2] += ((bits & 2u) ? re : -re) + ((bits & 32u) ? im : -im);
                    v[3] += ((bits & 4u) ? re : -re) + ((bits & 64u) ? im : -im);
                    v[4] += ((bits & 8u) ? re : -re) + ((bits & 128u) ? im : -im);
                    if (P.g_canon) reinterpret_cast<double2*>(P.g_canon)[k * (unsigned long long)V + i] = make_double2(re, im);
                }
                block_sum<5>(v, red, fb);   // its barrier also publishes the s_skip bits
                if (tid == 0) {
                    P.F_norm[k] = v[0] / ((double)DIM * (double)V);
                    P.sweeps[k] = tL;
                    P.status[k] = (uint8_t)((mxL ? 1 : 0) | (s_skip[L] ? 2 : 0));
                    reinterpret_cast<double4*>(P.sig)[k] =
                        make_double4(v[1] / (double)V, v[2] / (double)V, v[3] / (double)V, v[4] / (double)V);
                }
            }
            // the next start for lane L
            if (tid == 0) s_k = atomicAdd(P.counter, 1ull);
            __syncthreads();
            const unsigned long long k = s_k;
            if (k < P.n_starts) {
                const uint64_t s = P.start_ids ? P.start_ids[k] : P.first_start + k;
                double2* En = rows(eb ^ 1);   // where the next even half-sweep looks for its own sites
                for (int i = tid; i < V; i += kThreads) {   // a2: Philox counter (site, start lo, start hi, 0)
                    const u32x4 r = philox((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 0u, (uint32_t)P.seed,
                                           (uint32_t)(P.seed >> 32));
                    double sn, cs;
                    sincospi(unit_interval_pm1(r.x, r.y), &sn, &cs);
                    (parity_of<DIM>(D, i) ? A0 : En)[(size_t)i * 32 + L] = make_double2(cs, sn);
                }
                if (tid == 0) {
                    s_pos[L] = k;
                    s_skip[L] = 0u;
                }
                if (lane == L) {
                    active = true;
                    fresh = true;   // a new start begins with its even half-sweep
                    t = 0;
                    skipped = false;
                }
            } else if (lane == L) {
                active = false;
            }
            __syncthreads();
        }
        if (__ballot_sync(FULL, active) == 0) break;   // every warp holds the same lane states

        // ---------------------------------------------------------- odd half-sweep (second half of sweep t+1)
        {
            const bool commit = active && !fresh;
            const double2* E = rows(eb ^ 1);   // the values written by the last even half-sweep
            accO = 0.0;
            if constexpr (IDX::kBlocksN > 0) {
                accO = half_sweep_blocks<DIM, IDX::kBlocksN, 1, W1>(D, A0, A0, E, warp, lane, P.k2, commit, skipped);
            } else {
                for (int r = warp; r < half; r += kWarps) {
                    int i, jf[DIM], jb[DIM];
                    IDX::locate(D, 1, r, i, jf, jb);
                    double wr, wi;
                    neighbour_sum<DIM>(D, E, i, jf, jb, lane, wr, wi);
                    double2* own = A0 + (size_t)i * 32 + lane;
                    bool sk = false;
                    // own rows are read and written once per half-sweep: streaming hints keep L1 for the neighbour rows
                    const double2 gn = site_update<W1>(__ldcs(own), wr, wi, P.k2, sk);
                    if (commit) {
                        __stcs(own, gn);
                        const double dl = fma(gn.y, wr, -gn.x * wi);   // Delta_i = Im(g_i conj w_i) after the update
                        accO = fma(dl, dl, accO);
                        skipped |= sk;
                    }
                }
            }
            if (commit) ++t;
            fresh = false;
            eb ^= 1;
        }
        __syncthreads();

        // ---------------------------------------------------------- even half-sweep (first half of sweep t+1)
        double accE = 0.0;
        {
            const double2* E = rows(eb);
            double2* En = rows(eb ^ 1);
            if constexpr (IDX::kBlocksN > 0) {
                accE = half_sweep_blocks<DIM, IDX::kBlocksN, 0, W1>(D, E, En, A0, warp, lane, P.k2, active, skipped);
            } else {
                for (int r = warp; r < half; r += kWarps) {
                    int i, jf[DIM], jb[DIM];
                    IDX::locate(D, 0, r, i, jf, jb);
                    double wr, wi;
                    neighbour_sum<DIM>(D, A0, i, jf, jb, lane, wr, wi);
                    const double2 g = __ldcs(E + (size_t)i * 32 + lane);
                    const double dl = fma(g.y, wr, -g.x * wi);   // Delta_i of the field after sweep t
                    accE = fma(dl, dl, accE);
                    bool sk = false;
                    const double2 gn = site_update<W1>(g, wr, wi, P.k2, sk);
                    if (active) {
                        __stcs(En + (size_t)i * 32 + lane, gn);
                        skipped |= sk;
                    }
                }
            }
        }
        // a4: gauge precision of the field after sweep t (R5), fixed summation order over the warps
        sred[rb][warp][lane] = accE + accO;
        __syncthreads();
        double S = 0.0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) S += sred[rb][w][lane];
        rb ^= 1;
        const bool conv = active && t > 0 && (t % P.check_every == 0) && (S / (double)V < P.eps);
        maxed = active && !conv && t == P.max_sweeps;
        dumpm = __ballot_sync(FULL, conv || maxed);
        need = dumpm;
    }
}

// ---------------------------------------------------------------------------------------------------------
// Lattices with odd extents (3^4, 5x3x2, ...): the same lane-per-start layout, one small CTA (4 warps) per team, the
// update phases of reading R3 (parity, then level) from the orbit's tables with a CTA barrier after each, and the
// gauge precision from a separate pass over the post-sweep field (on an odd ring a same-parity neighbour may still
// move after w_i was formed, so the fused measure of the even lattices is not exact here: R5).  A team's field
// (V x 512 bytes: 41 KB at 3^4) stays in L1; four teams share an SM.
// ---------------------------------------------------------------------------------------------------------
constexpr int kPhasedThreads = 128;
constexpr int kPhasedWarps = kPhasedThreads / 32;

template <int DIM, bool W1, bool SMEM>
__global__ void __launch_bounds__(kPhasedThreads, 4) relax_phased_kernel(const StreamParams P) {
    constexpr unsigned FULL = 0xffffffffu;
    __shared__ double red[2][kPhasedWarps][5];
    __shared__ double sred[2][kPhasedWarps][32];
    __shared__ unsigned long long s_pos[32];
    __shared__ unsigned s_skip[32];
    __shared__ unsigned long long s_k;
    const OrbitDev& D = P.D;
    const int V = D.V;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // the team's field [V][32 starts]: in shared memory when four teams fit an SM (V <= 110: 3^4), else in the workspace (L1)
    extern __shared__ __align__(16) unsigned char phased_smem[];
    double2* const A = SMEM ? reinterpret_cast<double2*>(phased_smem) : P.team_buf + (size_t)blockIdx.x * V * 32;

    bool active = false, maxed = false, skipped = false;
    int t = 0, rb = 0, fb = 0;
    unsigned need = FULL, dumpm = 0;

    auto sum5 = [&](double (&v)[5]) {   // CTA sum, same result in every thread, fixed order
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
            for (int q = 0; q < 5; ++q) v[q] += __shfl_down_sync(FULL, v[q], o);
        if (lane == 0)
#pragma unroll
            for (int q = 0; q < 5; ++q) red[fb][warp][q] = v[q];
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            double sacc = 0.0;
            for (int w = 0; w < kPhasedWarps; ++w) sacc += red[fb][w][q];
            v[q] = sacc;
        }
        fb ^= 1;
    };

    for (;;) {
        // ---------------------------------------------------------- service (CTA-uniform): finalise, refill
        for (unsigned m = need; m; m &= m - 1) {
            const int L = __ffs(m) - 1;
            if ((dumpm >> L) & 1u) {   // a5, a6 for the start of lane L
                if (skipped) atomicOr(&s_skip[lane], 1u);
                const int tL = __shfl_sync(FULL, t, L);
                const int mxL = __shfl_sync(FULL, maxed ? 1 : 0, L);
                const unsigned long long k = s_pos[L];
                const double2 c = A[(size_t)(V - 1) * 32 + L];
                double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
                for (int i = tid; i < V; i += kPhasedThreads) {
                    const double2 gi = A[(size_t)i * 32 + L];
#pragma unroll
                    for (int mu = 0; mu < DIM; ++mu) {   // F = sum Re(g_i U_{i,mu} conj g_{i+mu})   (Eq. 3)
                        const double2 u = __ldg(D.U + i * DIM + mu);
                        const double2 gj = A[(size_t)__ldg(D.fwd + i * DIM + mu) * 32 + L];
                        const double ar = fma(gi.x, u.x, -gi.y * u.y), ai = fma(gi.x, u.y, gi.y * u.x);
                        v[0] += fma(ar, gj.x, ai * gj.y);
                    }
                    const double re = fma(gi.x, c.x, gi.y * c.y);   // g~ = g conj(g_{V-1})
                    const double im = fma(gi.y, c.x, -gi.x * c.y);
                    const unsigned bits = __ldg(D.sgn + i);
                    v[1] += ((bits & 1u) ? re : -re) + ((bits & 16u) ? im : -im);
                    v[2] += ((bits & 2u) ? re : -re) + ((bits & 32u) ? im : -im);
                    v[3] += ((bits & 4u) ? re : -re) + ((bits & 64u) ? im : -im);
                    v[4] += ((bits & 8u) ? re : -re) + ((bits & 128u) ? im : -im);
                    if (P.g_canon) reinterpret_cast<double2*>(P.g_canon)[k * (unsigned long long)V + i] = make_double2(re, im);
                }
                sum5(v);   // its barrier also publishes the s_skip bits
                if (tid == 0) {
                    P.F_norm[k] = v[0] / ((double)DIM * (double)V);
                    P.sweeps[k] = tL;
                    P.status[k] = (uint8_t)((mxL ? 1 : 0) | (s_skip[L] ? 2 : 0));
                    reinterpret_cast<double4*>(P.sig)[k] =
                        make_double4(v[1] / (double)V, v[2] / (double)V, v[3] / (double)V, v[4] / (double)V);
                }
            }
            if (tid == 0) s_k = atomicAdd(P.counter, 1ull);
            __syncthreads();
            const unsigned long long k = s_k;
            if (k < P.n_starts) {
                const uint64_t s = P.start_ids ? P.start_ids[k] : P.first_start + k;
                for (int i = tid; i < V; i += kPhasedThreads) {   // a2
                    const u32x4 r = philox((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 0u, (uint32_t)P.seed,
                                           (uint32_t)(P.seed >> 32));
                    double sn, cs;
                    sincospi(unit_interval_pm1(r.x, r.y), &sn, &cs);
                    A[(size_t)i * 32 + L] = make_double2(cs, sn);
                }
                if (tid == 0) {
                    s_pos[L] = k;
                    s_skip[L] = 0u;
                }
                if (lane == L) {
                    active = true;
                    t = 0;
                    skipped = false;
                }
            } else if (lane == L) {
                active = false;
            }
            __syncthreads();
        }
        if (__ballot_sync(FULL, active) == 0) break;   // every warp holds the same lane states

        // ---------------------------------------------------------- one sweep: the phases of R3, in place
        // accL: sum of Delta_i^2, taken right after the update, over the sites all of whose neighbours were updated
        // before them in this sweep (D.fin): for these it is the Delta of the post-sweep field, so accL summed over the
        // CTA is a LOWER BOUND of the gauge precision sum (with over-relaxation it is not zero: the update overshoots).
        double accL = 0.0;
        for (int p = 0; p < D.n_phases; ++p) {
            const int q1 = D.phase_off[p + 1];
            for (int q = D.phase_off[p] + warp; q < q1; q += kPhasedWarps) {
                int i, jf[DIM], jb[DIM];
                i = __ldg(D.order + q);
#pragma unroll
                for (int mu = 0; mu < DIM; ++mu) {
                    jf[mu] = __ldg(D.fwd + i * DIM + mu);
                    jb[mu] = __ldg(D.bwd + i * DIM + mu);
                }
                double wr, wi;
                neighbour_sum<DIM>(D, A, i, jf, jb, lane, wr, wi);
                double2* own = A + (size_t)i * 32 + lane;
                bool sk = false;
                const double2 gn = site_update<W1>(*own, wr, wi, P.k2, sk);
                if (active) {
                    *own = gn;
                    skipped |= sk;
                }
                if (__ldg(D.fin + i)) {   // warp-uniform
                    const double dl = fma(gn.y, wr, -gn.x * wi);
                    accL = fma(dl, dl, accL);
                }
            }
            __syncthreads();
        }
        if (active) ++t;

        // ---------------------------------------------------------- a4: gauge precision of the post-sweep field
        // The full pass over the field (a second neighbour sum per site) is needed only if some lane that is tested at
        // this sweep may pass: its lower bound is below 2 eps V (the factor 2 keeps rounding differences between the two
        // sums out of the decision).  Otherwise no lane can stop and the pass is skipped -- the decision is unchanged.
        sred[rb][warp][lane] = accL;
        __syncthreads();
        double Lsum = 0.0;
#pragma unroll
        for (int w = 0; w < kPhasedWarps; ++w) Lsum += sred[rb][w][lane];
        rb ^= 1;
        const bool tested = active && (t % P.check_every == 0);
#ifdef U1GF_PHASED_ALWAYS_FULL   // knob: the full gauge-precision pass after every sweep (what the lower bound saves)
        const bool may_pass = true;
#elif defined(U1GF_PHASED_NEVER_FULL)   // ablation knob (wrong results: nothing ever converges)
        const bool may_pass = false;
#else
        const bool may_pass = tested && !(Lsum / (double)V >= 2.0 * P.eps);
#endif
        double S = 0.0;
        if (__syncthreads_or(may_pass ? 1 : 0)) {
            double acc = 0.0;
            for (int i = warp; i < V; i += kPhasedWarps) {
                int jf[DIM], jb[DIM];
#pragma unroll
                for (int mu = 0; mu < DIM; ++mu) {
                    jf[mu] = __ldg(D.fwd + i * DIM + mu);
                    jb[mu] = __ldg(D.bwd + i * DIM + mu);
                }
                double wr, wi;
                neighbour_sum<DIM>(D, A, i, jf, jb, lane, wr, wi);
                const double2 g = A[(size_t)i * 32 + lane];
                const double dl = fma(g.y, wr, -g.x * wi);   // Delta_i = Im(g_i conj w_i)
                acc = fma(dl, dl, acc);
            }
            sred[rb][warp][lane] = acc;
            __syncthreads();
#pragma unroll
            for (int w = 0; w < kPhasedWarps; ++w) S += sred[rb][w][lane];
            rb ^= 1;
        } else {
            S = 2.0 * P.eps * (double)V;   // not below eps V for any tested lane
        }
        const bool conv = active && (t % P.check_every == 0) && (S / (double)V < P.eps);
        maxed = active && !conv && t == P.max_sweeps;
        dumpm = __ballot_sync(FULL, conv || maxed);
        need = dumpm;
    }
}

template <int DIM, bool W1, bool SMEM>
int launch_phased_k(const u1gf_orbit* o, const RelaxArgs& a, StreamParams& P, cudaStream_t st) {
    auto kern = relax_phased_kernel<DIM, W1, SMEM>;
    const size_t smem = SMEM ? (size_t)o->dev.V * 32 * sizeof(double2) : 0;
    if (SMEM) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    else cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 5);
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kPhasedThreads, smem) != cudaSuccess) per_sm = 0;
    unsigned long long teams = (unsigned long long)per_sm * (unsigned long long)o->sm_count;
    const unsigned long long batches = (a.n_starts + 31) / 32;
    if (teams > batches) teams = batches;
    if (teams > 4ull * (unsigned long long)o->sm_count) teams = 4ull * (unsigned long long)o->sm_count;   // workspace bound
    if (teams < 1) return fail(U1GF_ECUDA, "phased relaxation kernel does not fit on an SM");
    const size_t bytes = 256 + (SMEM ? 0 : (size_t)teams * (size_t)o->dev.V * 32 * sizeof(double2));
    U1GF_CUDA(cudaMemsetAsync(a.workspace, 0, bytes, st));
    kern<<<(unsigned)teams, kPhasedThreads, smem, st>>>(P);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    return U1GF_OK;
}

template <int DIM, bool W1, class IDX>
int launch_k(const u1gf_orbit* o, const RelaxArgs& a, StreamParams& P, cudaStream_t st) {
    auto kern = relax_stream_kernel<DIM, W1, IDX>;
    cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 5);   // percent: the rest is L1 for the rows
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, 0) != cudaSuccess) per_sm = 0;
    unsigned long long teams = (unsigned long long)per_sm * (unsigned long long)o->sm_count;
    const unsigned long long batches = (a.n_starts + 31) / 32;
    if (teams > batches) teams = batches;
    if (teams > 2ull * (unsigned long long)o->sm_count) teams = 2ull * (unsigned long long)o->sm_count;   // workspace bound
    if (teams < 1) return fail(U1GF_ECUDA, "streamed relaxation kernel does not fit on an SM");
    // counter and team buffers start from zero (an idle lane then reads a null field, not stale bits)
    const size_t bytes = 256 + (size_t)teams * 2 * (size_t)o->dev.V * 32 * sizeof(double2);
    U1GF_CUDA(cudaMemsetAsync(a.workspace, 0, bytes, st));
    kern<<<(unsigned)teams, kThreads, 0, st>>>(P);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    return U1GF_OK;
}

template <int DIM, class IDX>
int launch_w(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st) {
    const bool w1 = a.omega == 1.0;
    StreamParams P;
    P.seed = a.seed; P.first_start = a.first_start; P.n_starts = a.n_starts; P.start_ids = a.start_ids;
    P.k2 = w1 ? 0.0 : a.omega / (1.0 - a.omega); P.eps = a.eps;
    P.max_sweeps = a.max_sweeps; P.check_every = a.check_every;
    P.F_norm = a.F_norm; P.sweeps = a.sweeps; P.status = a.status; P.sig = a.sig; P.g_canon = a.g_canon;
    P.counter = (unsigned long long*)a.workspace;
    P.team_buf = (double2*)((char*)a.workspace + 256);
    P.D = o->dev;
    return w1 ? launch_k<DIM, true, IDX>(o, a, P, st) : launch_k<DIM, false, IDX>(o, a, P, st);
}

template <int DIM>
bool cubic(const u1gf_orbit* o, int n) {
    for (int mu = 0; mu < DIM; ++mu)
        if (o->dev.ext[mu] != n) return false;
    return true;
}

template <int DIM>
int launch_phased(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st) {
    const bool w1 = a.omega == 1.0;
    StreamParams P;
    P.seed = a.seed; P.first_start = a.first_start; P.n_starts = a.n_starts; P.start_ids = a.start_ids;
    P.k2 = w1 ? 0.0 : a.omega / (1.0 - a.omega); P.eps = a.eps;
    P.max_sweeps = a.max_sweeps; P.check_every = a.check_every;
    P.F_norm = a.F_norm; P.sweeps = a.sweeps; P.status = a.status; P.sig = a.sig; P.g_canon = a.g_canon;
    P.counter = (unsigned long long*)a.workspace;
    P.team_buf = (double2*)((char*)a.workspace + 256);
    P.D = o->dev;
#ifndef U1GF_PHASED_SMEM_MAXV
#define U1GF_PHASED_SMEM_MAXV 110   // 4 teams x V x 512 bytes within the shared memory of an SM
#endif
    if (o->dev.V <= U1GF_PHASED_SMEM_MAXV)
        return w1 ? launch_phased_k<DIM, true, true>(o, a, P, st) : launch_phased_k<DIM, false, true>(o, a, P, st);
    return w1 ? launch_phased_k<DIM, true, false>(o, a, P, st) : launch_phased_k<DIM, false, false>(o, a, P, st);
}

template <int DIM>
int launch(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st) {
    if (!o->dev.all_even) return launch_phased<DIM>(o, a, st);
    if (DIM >= 2) {
        if (cubic<DIM>(o, 6)) return launch_w<DIM, Cubic<DIM, 6>>(o, a, st);
        if (cubic<DIM>(o, 8)) return launch_w<DIM, Cubic<DIM, 8>>(o, a, st);
        if (DIM <= 3 && cubic<DIM>(o, 10)) return launch_w<DIM, Cubic<DIM, 10>>(o, a, st);
    }
    return launch_w<DIM, Tables<DIM>>(o, a, st);
}

}  // namespace

// every extent even (two-colour checkerboard); chosen automatically from 512 sites up, where a team's field no longer
// fits on chip and the generic kernel's per-start link traffic dominates
bool stream_supported(const u1gf_orbit* o) { return o->dev.d >= 1 && o->dev.d <= 4; }
// automatic choice: all-even lattices from 1024 sites up (the fused two-colour kernel; measured against the generic
// kernel: 6^4 302 vs 732 ms, 8^4 960 vs 1777 ms, but 8^3 41 vs 29 ms and 12^2 14 vs 13 ms -- below about a thousand
// sites the two barriers per sweep outweigh the shared link reads), lattices with an odd extent from 64 sites up (the
// phased kernel; 3^4 = 81: 87 vs 320 ms)
bool stream_preferred(const u1gf_orbit* o) {
    return stream_supported(o) && (o->dev.all_even ? o->dev.V >= 1024 : o->dev.V >= 64);
}

size_t stream_workspace_bytes(const u1gf_orbit* o, uint64_t n) {
    // upper bound on the teams of a launch: 2 CTAs per SM with two buffers each (even lattices) or 4 CTAs per SM with
    // one buffer (odd extents): the same bytes; never more than the batches of 32 starts
    unsigned long long teams = 2ull * (unsigned long long)o->sm_count;
    const unsigned long long batches = (n + 31) / 32;
    if (teams > batches) teams = batches;
    if (teams < 1) teams = 1;
    return 256 + (size_t)teams * 2 * (size_t)o->dev.V * 32 * sizeof(double2);
}

int stream_relax(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st) {
    switch (o->dev.d) {
        case 1: return launch<1>(o, a, st);
        case 2: return launch<2>(o, a, st);
        case 3: return launch<3>(o, a, st);
        default: return launch<4>(o, a, st);
    }
}

}  // namespace u1gf
