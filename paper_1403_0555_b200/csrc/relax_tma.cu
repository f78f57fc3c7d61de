// relax_tma.cu -- TMA-staged streamed "lane per start" relaxation kernel for the large 4D lattices (6^4, 8^4):
// north_star's "larger lattices stream parity halves through TMA-staged tiles with coalesced 128-bit loads".
//
// As in relax_stream.cu the gauge field of a team of 32 starts lives in HBM / L2, one 512-byte row per site (lane =
// start), and lane l of every warp works on start l, so a link is read once per 32 site updates.  What changes is how
// the rows reach the SM.  The LDG kernel is bound by the latency of its dependent, register-staged row loads (ncu:
// 6.9 long-scoreboard stalls per issued instruction, DRAM 23 % busy); here the rows of the OTHER parity -- the eight
// neighbours of every site -- are brought into shared memory by bulk asynchronous copies (cp.async.bulk, SASS UBLKCP)
// that a producer warp issues several tiles ahead, completion counted by mbarriers, and the consumer warps read them
// with conflict-free LDS.128.  The data in flight sits in shared memory (about 100 KB per SM), not in registers.
//
// Layout of a team's field (workspace): three arrays O (odd sites), E (even sites) and SV (the pre-update even values
// of the lanes that may stop at this sweep, see the kernel), each [sheet = x3*N + x2][x1][k][32 starts] double2, where
// the half-line (x1, x2, x3) of parity p holds the sites x0 = 2k + ((p + x1 + x2 + x3) & 1), k = 0 .. N/2-1.  A
// "half-sheet" (all x0, x1 of one parity at fixed x2, x3) is one contiguous block of N * N/2 rows = 16 KB at N = 8,
// 9 KB at N = 6: the unit of a bulk copy.
//
// A half-sweep walks the sheets in order (x3 outer, x2 inner), one step per sheet.  For the sites of parity p in sheet
// (x2, x3) the neighbours along x0 and x1 are in the other-parity half-sheet (x2, x3), those along x2 in the
// half-sheets (x2 -+ 1, x3) -- these three slide through a window of RW slots as x2 advances, so each is fetched
// once per layer (N + 2 fetches for N steps) -- and those along x3 in the half-sheets (x2, x3 -+ 1), fetched per step
// into a ring of ST stages together with the step's links ([site][8] double2: U_{i,mu}, U_{i-mu,mu}).  Per site
// update: 16 B (window) * (N+2)/N + 32 B (x3 neighbours) + 16 B own row read + 16 B written = 84 B between L2 and
// the SM; at 8^4 the 48 B that are not re-reads come from HBM (the x3 re-reads hit L2; own rows carry streaming
// hints), at 6^4 the 96 MB that 148 teams cycle through stay in L2.  The own row of a site is private to the thread
// that updates it (same warp, same lane every sweep): it is read by a plain coalesced load one step ahead and written
// back from registers.  Measured bounds and what was tried: DESIGN.md section 7.4, profiles/r02_ablations.md.
//
// Arithmetic of a site update, stop rule (R5), lane-level refill and finalisation are those of relax_stream.cu.
#include "u1gf_internal.h"

namespace u1gf {
namespace {

struct TmaParams {
    uint64_t seed, first_start, n_starts;
    const uint64_t* start_ids;
    double k2, eps;   // k2 = omega / (1 - omega) (unused when omega == 1)
    int max_sweeps, check_every;
    double* F_norm;
    int32_t* sweeps;
    uint8_t* status;
    double* sig;
    double* g_canon;
    double2* team_buf;             // [teams][3][V/2][32]: O, E, SV
    const double2* lnk;            // [2][V/2][8]: links in row order, forward U_{i,mu} then backward U_{i-mu,mu}
    unsigned long long* counter;   // next start position to hand out
    OrbitDev D;
};

template <int N>
struct TG {
    static constexpr int H = N / 2;            // rows of a half-line
    static constexpr int SITES = N * H;        // sites of one parity in a sheet = sites per step
#ifndef U1GF_TMA_SPW8
#define U1GF_TMA_SPW8 4
#endif
#ifndef U1GF_TMA_SPW6
#define U1GF_TMA_SPW6 3
#endif
    static constexpr int SPW = N == 8 ? U1GF_TMA_SPW8 : U1GF_TMA_SPW6;   // sites per consumer warp and step (knobs: 8^4: 4, 2, 1; 6^4: 3, 1)
#ifndef U1GF_TMA_GRP6
#define U1GF_TMA_GRP6 1
#endif
    static constexpr int NGRP = N >= 8 ? 1 : U1GF_TMA_GRP6;   // groups of consumer warps; group r works on the steps g = r (mod NGRP), so NGRP steps are in progress at a time
    static constexpr int CWG = SITES / SPW;    // consumer warps of a group (8^4: 8 x a half-line of 4 sites, 6^4: 6 x a half-line of 3)
    static constexpr int CW = CWG * NGRP;      // consumer warps
    static constexpr int THREADS = (CW + 1) * 32;   // + the producer warp
    static constexpr int V = N * N * N * N, HALF = V / 2;
    static constexpr int NS = N * N;           // steps per half-sweep
    static constexpr int WL = N * (N + 2);     // window fetches per half-sweep
#ifndef U1GF_TMA_ST6
#define U1GF_TMA_ST6 4
#endif
#ifndef U1GF_TMA_RW6
#define U1GF_TMA_RW6 6
#endif
#ifndef U1GF_TMA_LA6
#define U1GF_TMA_LA6 2
#endif
    static constexpr int RW = N >= 8 ? 6 : U1GF_TMA_RW6;          // window slots
    static constexpr int ST = N >= 8 ? 3 : U1GF_TMA_ST6;          // stages of the x3-neighbour / link ring
    static constexpr int LA = N >= 8 ? 2 : U1GF_TMA_LA6;          // steps the window fetches run ahead
    static constexpr unsigned HSMOD = 4 * RW * ST;
    static constexpr unsigned SHEET_B = SITES * 512, LNK_B = SITES * 128;
    static constexpr size_t off_win = 0;
    static constexpr size_t off_x3 = off_win + (size_t)RW * SHEET_B;
    static constexpr size_t off_lnk = off_x3 + (size_t)ST * 2 * SHEET_B;
    static constexpr size_t off_bar = off_lnk + (size_t)ST * LNK_B;           // fullW[RW], fullS[ST], empty[ST]
    static constexpr size_t off_sred = off_bar + (size_t)(RW + 2 * ST) * 8 + 8;
    static constexpr size_t off_red = off_sred + (size_t)(5 * CW + 1) * 32 * 8;   // [2][CW][32] sweep sums, [CW][32] odd sums, [2][CW][32] F sums, [32] F of the lanes that stop
    static constexpr size_t off_pos = off_red + (size_t)2 * (CW + 1) * 5 * 8;
    static constexpr size_t off_skip = off_pos + 32 * 8;
    static constexpr size_t smem_bytes = off_skip + 32 * 4 + 16;
    static_assert(SITES % SPW == 0 && N % 2 == 0 && (N * N) % (2 * NGRP) == 0 && ST > NGRP, "geometry");
};

// ---------------------------------------------------------------------------------------------------------
// mbarrier / bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk)
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// global -> shared bulk copy (TMA engine), completion reported to the mbarrier in bytes
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
// orders this thread's earlier generic-proxy accesses (global stores of rows) before later async-proxy ones (bulk copies)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// sum over the CTA of NV per-thread values, same result in every thread, fixed order (deterministic)
template <int NV, int NWARPS>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* red, int& buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int q = 0; q < NV; ++q) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* r = red + (size_t)buf * NWARPS * NV;
    if (lane == 0)
#pragma unroll
        for (int q = 0; q < NV; ++q) r[warp * NV + q] = v[q];
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NV; ++q) {
        double s = 0.0;
        for (int w = 0; w < NWARPS; ++w) s += r[w * NV + q];
        v[q] = s;
    }
    buf ^= 1;
}

// a3 for one site of one start: g <- normalise((1-omega) g + omega w/|w|) (R2), the 8d+20 form of
// relax_lanes.cu (h' = g + (k2/|w|) w = h/(1-omega), second-order rsqrt polish); W1: omega == 1, g <- w/|w|.
// R6 (|w|^2 < 1e-280: the site keeps its value) by selects, not a branch: the sites a warp updates in one step then
// form ONE basic block and ptxas interleaves their dependent chains (with the branch, each site ran alone and the warp
// issued one instruction every 5 cycles).
template <bool W1>
__device__ __forceinline__ double2 site_update(double2 g, double wr, double wi, double k2, bool& small) {
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
    // bit patterns of non-negative doubles are ordered like the numbers
    small = (unsigned long long)__double_as_longlong(nw) < (unsigned long long)__double_as_longlong(1e-280);
    gn.x = small ? g.x : gn.x;
    gn.y = small ? g.y : gn.y;
    return gn;
}

// site index -> (parity, row inside the parity's array)
template <int N>
__device__ __forceinline__ void locate(int i, int& p, int& row) {
    const int x0 = i % N, l = i / N;
    const int x1 = l % N, x2 = (l / N) % N, x3 = l / (N * N);
    p = (x0 + x1 + x2 + x3) & 1;
    row = l * (N / 2) + (x0 >> 1);
}

#ifdef U1GF_TMA_PROF   // debugging knob: cycle counters of CTA 0 printed at the end of the kernel
__device__ unsigned long long g_prof[16];
#define PROF_T0() const long long prof_t0 = clock64()
#define PROF_ADD(k) if (blockIdx.x == 0 && lane == 0) atomicAdd(&g_prof[k], (unsigned long long)(clock64() - prof_t0))
#else
#define PROF_T0()
#define PROF_ADD(k)
#endif

template <int N>
struct Smem {
    unsigned win, x3, lnk, fullW, fullS, empty;   // shared-space addresses
    const unsigned char* base;                    // the dynamic shared memory as a generic pointer
};

// One half-sweep of parity PAR.  src / dst: rows of parity PAR before / after the update (the same array); save: where
// the lanes with `cand` set keep their pre-update values (even half-sweep); oth: rows of the other parity; lnk: links of the parity-PAR sites in row order.  `hs` counts the
// half-sweeps of this CTA (the mbarrier phases follow from it).  Returns sum Delta_i^2 over this warp's sites for the
// lane's start: PAR == 0 measured before the update (field after the previous sweep), PAR == 1 after it.
template <int N, int PAR, bool W1>
__device__ __forceinline__ double half_sweep(const Smem<N>& S, const double2* src, double2* dst, double2* save,
                                             const double2* __restrict__ oth, const double2* __restrict__ lnk, unsigned hs,
                                             int warp, int lane, double k2, bool commit, bool cand, bool& skipped, double& accF) {
    using G = TG<N>;
    constexpr int H = G::H, SITES = G::SITES, SPW = G::SPW, CW = G::CW, NS = G::NS, WL = G::WL, RW = G::RW, ST = G::ST;
    const unsigned step0 = hs * NS, wl0 = hs * WL;
    double acc = 0.0;
    // (the caller has put fence.proxy.async + a CTA barrier in front: rows written by this CTA with ordinary stores --
    // last half-sweep, refill -- must be visible to the bulk copies)
    if (warp == CW) {
        // ------------------------------------------------------------------ producer: one lane issues every bulk copy
        if (lane == 0) {
            int nw = 0, nsl = 0;   // next window fetch / next stage fetch of this half-sweep
            for (int g = 0; g < NS; ++g) {
                if (g > 0) {   // steps up to g-1 are finished by every consumer warp
                    const unsigned sg = step0 + g - 1;
                    PROF_T0();
                    mbar_wait(S.empty + (sg % ST) * 8, (sg / ST) & 1u);
                    PROF_ADD(0);
                }
                // x3 neighbours and links of the steps below g + ST: the stage of step s was last used by step s - ST
                while (nsl < NS && nsl < g + ST) {
                    const int x3 = nsl / N, x2 = nsl % N;
                    const unsigned sg = step0 + nsl, st = sg % ST, bar = S.fullS + st * 8;
#ifdef U1GF_TMA_ABL_NOX3   // ablation knob (wrong results): the x3 neighbours are not fetched (52 instead of 84 B per site update)
                    mbar_expect_tx(bar, G::LNK_B);
#else
                    mbar_expect_tx(bar, 2 * G::SHEET_B + G::LNK_B);
                    const int dn = ((x3 + N - 1) % N) * N + x2, up = ((x3 + 1) % N) * N + x2;
                    bulk_g2s(S.x3 + (st * 2 + 0) * G::SHEET_B, oth + (size_t)dn * SITES * 32, G::SHEET_B, bar);
                    bulk_g2s(S.x3 + (st * 2 + 1) * G::SHEET_B, oth + (size_t)up * SITES * 32, G::SHEET_B, bar);
#endif
                    bulk_g2s(S.lnk + st * G::LNK_B, lnk + (size_t)nsl * SITES * 8, G::LNK_B, bar);
                    ++nsl;
                }
                // window: fetch q of layer x3 is the half-sheet x2 = q - 1 (mod N); step (x3, x2) uses fetches x2, x2+1, x2+2
                const int gl = g + G::LA < NS ? g + G::LA : NS - 1;
                const int need = (gl / N) * (N + 2) + gl % N + 2;
                while (nw <= need) {
                    if (nw >= RW) {   // its slot was last used by fetch nw - RW, whose last reader is step min(q, N-1) of its layer
                        const int o = nw - RW, oq = o % (N + 2);
                        const int lu = (o / (N + 2)) * N + (oq < N - 1 ? oq : N - 1);
                        if (lu >= g) break;
                    }
                    const int x3 = nw / (N + 2), x2 = (nw % (N + 2) + N - 1) % N;
                    const unsigned gw = wl0 + nw, sl = gw % RW, bar = S.fullW + sl * 8;
                    mbar_expect_tx(bar, G::SHEET_B);
                    bulk_g2s(S.win + sl * G::SHEET_B, oth + (size_t)(x3 * N + x2) * SITES * 32, G::SHEET_B, bar);
                    ++nw;
                }
            }
        }
        __syncwarp();
        return 0.0;
    }

    // ---------------------------------------------------------------------- consumers: SPW sites per warp and step
    // Per-step bookkeeping is kept incremental and everything that depends only on the warp's sites is formed once:
    // with SPW sites per warp and step every instruction outside the site update is paid SPW times less often.
    // ordinary shared-memory loads (offsets from the start of the dynamic shared memory): the mbarrier waits are asm
    // statements with a memory clobber, so the compiler keeps these loads behind them and is otherwise free to schedule
    auto lds = [&](unsigned off) { return *reinterpret_cast<const double2*>(S.base + off); };
    constexpr bool LINE = SPW == H;   // a warp owns a whole half-line: its H rows of the other parity serve all x0 neighbours
    constexpr int NGRP = G::NGRP;
    const int grp = warp / G::CWG;                // this warp works on the steps g = grp, grp + NGRP, ...
    const int q0 = (warp % G::CWG) * SPW;         // first site of this warp inside a half-sheet, q = x1 * H + k
    const unsigned l16 = lane * 16;
    unsigned vF0[SPW][2], vB0[SPW][2], vF1[SPW], vB1[SPW], vQ[SPW];   // byte offsets inside a half-sheet (+ the lane's 16 bytes)
    unsigned vRow[LINE ? H : 1];
    int abase[SPW];
#pragma unroll
    for (int j = 0; j < SPW; ++j) {
        const int q = q0 + j, x1 = q / H, k = q % H;
        const int x1f = x1 + 1 == N ? 0 : x1 + 1, x1b = x1 == 0 ? N - 1 : x1 - 1;
#pragma unroll
        for (int a = 0; a < 2; ++a) {   // x0 = 2k + a
            const int kf = a ? (k + 1 == H ? 0 : k + 1) : k, kb = a ? k : (k == 0 ? H - 1 : k - 1);
            vF0[j][a] = (x1 * H + kf) * 512 + l16;
            vB0[j][a] = (x1 * H + kb) * 512 + l16;
        }
        vF1[j] = (x1f * H + k) * 512 + l16;
        vB1[j] = (x1b * H + k) * 512 + l16;
        vQ[j] = q * 512 + l16;
        abase[j] = (PAR + x1) & 1;
        if (LINE) vRow[LINE ? j : 0] = vQ[j];
    }
    double2 own[SPW], nxt[SPW];
    const double2* psrc = src + ((size_t)grp * SITES + q0) * 32 + lane;
    double2* pdst = dst + ((size_t)grp * SITES + q0) * 32 + lane;
#pragma unroll
    for (int j = 0; j < SPW; ++j) own[j] = __ldcs(psrc + j * 32);
    // ring positions of step 0: window fetch of the x2-1 half-sheet (slot, phase parity), stage (index, phase parity)
    unsigned sDn = wl0 % RW, pDn = (wl0 / RW) & 1u, st = step0 % ST, pst = (step0 / ST) & 1u;
    int x2 = 0, sp = 0;   // sp = (x2 + x3) & 1
    // the window advances by one fetch inside a layer and by three at a layer boundary (N + 2 fetches per layer)
    auto advance = [&]() {
        if (++st == ST) st = 0, pst ^= 1u;
        if (++x2 == N) {
            x2 = 0;   // x2: N-1 -> 0 and x3 + 1: the sheet parity stays
            sDn += 3;
        } else {
            sp ^= 1;
            sDn += 1;
        }
        if (sDn >= RW) sDn -= RW, pDn ^= 1u;
    };
    for (int r = 0; r < grp; ++r) advance();
    auto step = [&](int g, double2 (&own)[SPW], double2 (&nxt)[SPW]) {
        psrc += NGRP * SITES * 32;
        if (g + NGRP < NS) {
#pragma unroll
            for (int j = 0; j < SPW; ++j) nxt[j] = __ldcs(psrc + j * 32);
        }
        unsigned sC = sDn + 1, pC = pDn;
        if (sC == RW) sC = 0, pC ^= 1u;
        unsigned sUp = sC + 1, pUp = pC;
        if (sUp == RW) sUp = 0, pUp ^= 1u;
        PROF_T0();
        if (NGRP > 1 || x2 == 0) {   // first step of a layer: all three half-sheets are new; later ones were waited for as C / Up
            mbar_wait(S.fullW + sDn * 8, pDn);
            mbar_wait(S.fullW + sC * 8, pC);
        }
        mbar_wait(S.fullW + sUp * 8, pUp);
        mbar_wait(S.fullS + st * 8, pst);
        if (warp == 0) { PROF_ADD(1); }
        const unsigned bC = (unsigned)G::off_win + sC * G::SHEET_B, bDn2 = (unsigned)G::off_win + sDn * G::SHEET_B,
                       bUp2 = (unsigned)G::off_win + sUp * G::SHEET_B;
        const unsigned bDn3 = (unsigned)G::off_x3 + (st * 2) * G::SHEET_B, bUp3 = bDn3 + G::SHEET_B;
        const unsigned bL = (unsigned)G::off_lnk + st * G::LNK_B + q0 * 128;
        double2 cf[LINE ? H : 1];
        if (LINE) {   // cf[k] = row (k + a) mod H of the warp's line: x0+1 neighbour of site k, x0-1 neighbour of site k+1
            const int a = abase[0] ^ sp;
#pragma unroll
            for (int k = 0; k < H; ++k) cf[LINE ? k : 0] = lds(bC + (a ? vRow[LINE ? (k + 1) % H : 0] : vRow[LINE ? k : 0]));
        }
#pragma unroll
        for (int j = 0; j < SPW; ++j) {
            const int a = abase[j] ^ sp;
            double2 gf[4], gb[4], uf[4], ub[4];
            if (LINE) {
                gf[0] = cf[LINE ? j : 0];
                gb[0] = cf[LINE ? (j + H - 1) % H : 0];
            } else {
                gf[0] = lds(bC + (a ? vF0[j][1] : vF0[j][0]));
                gb[0] = lds(bC + (a ? vB0[j][1] : vB0[j][0]));
            }
            gf[1] = lds(bC + vF1[j]);
            gb[1] = lds(bC + vB1[j]);
            gf[2] = lds(bUp2 + vQ[j]);
            gb[2] = lds(bDn2 + vQ[j]);
            gf[3] = lds(bUp3 + vQ[j]);
            gb[3] = lds(bDn3 + vQ[j]);
#pragma unroll
            for (int mu = 0; mu < 4; ++mu) {
                uf[mu] = lds(bL + (j * 8 + mu) * 16);
                ub[mu] = lds(bL + (j * 8 + 4 + mu) * 16);
            }
            double wr = 0.0, wi = 0.0;
#pragma unroll
            for (int mu = 0; mu < 4; ++mu) {   // w_i = sum_mu [conj(U_{i,mu}) g_{i+mu} + U_{i-mu,mu} g_{i-mu}]  (= conj K_i, Eq. 5)
                wr = fma(uf[mu].x, gf[mu].x, wr);
                wi = fma(uf[mu].x, gf[mu].y, wi);
                wr = fma(uf[mu].y, gf[mu].y, wr);
                wi = fma(-uf[mu].y, gf[mu].x, wi);
                wr = fma(ub[mu].x, gb[mu].x, wr);
                wi = fma(ub[mu].x, gb[mu].y, wi);
                wr = fma(-ub[mu].y, gb[mu].y, wr);
                wi = fma(ub[mu].y, gb[mu].x, wi);
            }
            const double2 gi = own[j];
            if (PAR == 0) {
                const double dl = fma(gi.y, wr, -gi.x * wi);   // Delta_i of the field after sweep t
                acc = fma(dl, dl, acc);
                // a5: every link joins an even and an odd site, so the sum over the even sites of Re(g_i conj w_i) on the
                // field before this update is F = sum_{i,mu} Re(g_i U_{i,mu} conj g_{i+mu}) of the field after sweep t
                // (Eq. 3): two FMAs per even site instead of four gathered neighbours in the finalisation
                accF = fma(gi.x, wr, accF);
                accF = fma(gi.y, wi, accF);
            }
            bool sk;
            const double2 gn = site_update<W1>(gi, wr, wi, k2, sk);
            if (PAR == 0 && cand) save[(pdst - dst) + j * 32] = gi;   // R5: a lane that may stop keeps its pre-update value
            if (commit) __stcs(pdst + j * 32, gn);
            if (PAR == 1) {   // (a lane without commit drops the sum below)
                const double dl = fma(gn.y, wr, -gn.x * wi);   // Delta_i = Im(g_i conj w_i) after the update
                acc = fma(dl, dl, acc);
            }
            skipped |= sk && commit;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(S.empty + st * 8);   // this warp no longer reads the buffers of step g
        pdst += NGRP * SITES * 32;
#pragma unroll
        for (int r = 0; r < NGRP; ++r) advance();
    };
    // two steps per iteration: the rows fetched for the next step land in the other register set (no copies, so the
    // load has a whole step to arrive)
    for (int g = grp; g < NS; g += 2 * NGRP) {
        step(g, own, nxt);
        step(g + NGRP, nxt, own);
    }
    if (PAR == 1 && !commit) acc = 0.0;
    return acc;
}

template <int N, bool W1>
__global__ void __launch_bounds__(TG<N>::THREADS, 1) relax_tma_kernel(const TmaParams P) {
    using G = TG<N>;
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int V = G::V, HALF = G::HALF, CW = G::CW, NW = CW + 1, THREADS = G::THREADS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* sred = reinterpret_cast<double*>(smem_raw + G::off_sred);              // [2][CW][32]
    double* sredO = sred + 2 * CW * 32;                                            // [CW][32]
    double* sredF = sredO + CW * 32;                                               // [2][CW][32]
    double* s_F = sredF + 2 * CW * 32;                                             // [32]
    double* red = reinterpret_cast<double*>(smem_raw + G::off_red);                // [2][NW][5]
    unsigned long long* s_pos = reinterpret_cast<unsigned long long*>(smem_raw + G::off_pos);
    unsigned* s_skip = reinterpret_cast<unsigned*>(smem_raw + G::off_skip);
    __shared__ unsigned long long s_k;
    const OrbitDev& D = P.D;
    const int tid = threadIdx.x, lane = tid & 31, warp = __shfl_sync(FULL, tid >> 5, 0);
    double2* const O = P.team_buf + (size_t)blockIdx.x * 3 * HALF * 32;
    double2* const E = O + (size_t)HALF * 32;
    // Stop rule R5: the decision on sweep t needs the even-site Delta formed by the even half-sweep of sweep t+1, and a
    // start that stops must keep the even values from BEFORE that half-sweep.  The LDG kernel double-buffers the even
    // rows for this; here only the lanes that can stop at this sweep -- the odd part of the gauge precision is already
    // below eps (a necessary condition), or max_sweeps is reached -- save their old even values to SV (16-byte stores of
    // one or two lanes per row), and the even rows are updated in place.  A team then cycles through 2 x V/2 rows
    // instead of 3: 648 KB at 6^4, 96 MB over 148 teams, which stays in the 126 MB L2.
    double2* const SV = E + (size_t)HALF * 32;

    Smem<N> S;
    S.base = smem_raw;
    S.win = smem_u32(smem_raw + G::off_win);
    S.x3 = smem_u32(smem_raw + G::off_x3);
    S.lnk = smem_u32(smem_raw + G::off_lnk);
    S.fullW = smem_u32(smem_raw + G::off_bar);
    S.fullS = S.fullW + G::RW * 8;
    S.empty = S.fullS + G::ST * 8;
    if (tid == 0) {
        for (int s = 0; s < G::RW; ++s) mbar_init(S.fullW + s * 8, 1);
        for (int s = 0; s < G::ST; ++s) {
            mbar_init(S.fullS + s * 8, 1);
            mbar_init(S.empty + s * 8, G::CWG);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    bool active = false, fresh = false, maxed = false, skipped = false;
    int t = 0, rb = 0, fb = 0;
    unsigned hs = 0;
    double accO = 0.0;
    unsigned need = FULL, dumpm = 0;   // first pass: every lane needs a start, nothing to finalise

    for (;;) {
        // ---------------------------------------------------------- service (CTA-uniform): finalise, refill
#ifdef U1GF_TMA_PROF
        const long long prof_s0 = clock64();
#endif
        for (unsigned m = need; m; m &= m - 1) {
            const int L = __ffs(m) - 1;
            if ((dumpm >> L) & 1u) {
                // a5, a6 for the start of lane L: even rows before the last even half-sweep (saved in SV), odd rows O
                if (skipped) atomicOr(&s_skip[lane], 1u);
                const int tL = __shfl_sync(FULL, t, L);
                const int mxL = __shfl_sync(FULL, maxed ? 1 : 0, L);
                const unsigned long long k = s_pos[L];
                int pc, rc;
                locate<N>(V - 1, pc, rc);
                const double2 c = (pc ? O : SV)[(size_t)rc * 32 + L];
                double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#ifdef U1GF_TMA_PROF
                const long long prof_f0 = clock64();
#endif
                for (int i = tid; i < V; i += THREADS) {
                    int pi, ri;
                    locate<N>(i, pi, ri);
                    const double2 gi = (pi ? O : SV)[(size_t)ri * 32 + L];
                    const double re = fma(gi.x, c.x, gi.y * c.y);   // g~ = g conj(g_{V-1})
                    const double im = fma(gi.y, c.x, -gi.x * c.y);
                    const unsigned bits = __ldg(D.sgn + i);
                    v[1] += ((bits & 1u) ? re : -re) + ((bits & 16u) ? im : -im);
                    v[2] += ((bits & 2u) ? re : -re) + ((bits & 32u) ? im : -im);
                    v[3] += ((bits & 4u) ? re : -re) + ((bits & 64u) ? im : -im);
                    v[4] += ((bits & 8u) ? re : -re) + ((bits & 128u) ? im : -im);
                    if (P.g_canon) reinterpret_cast<double2*>(P.g_canon)[k * (unsigned long long)V + i] = make_double2(re, im);
                }
#ifdef U1GF_TMA_PROF
                if (blockIdx.x == 0 && tid == 0) atomicAdd(&g_prof[4], (unsigned long long)(clock64() - prof_f0));
#endif
                block_sum<5, NW>(v, red, fb);   // its barrier also publishes the s_skip bits
                if (tid == 0) {
                    P.F_norm[k] = s_F[L] / (4.0 * (double)V);   // a5 came out of the last even half-sweep
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
#ifdef U1GF_TMA_PROF
                const long long prof_r0 = clock64();
#endif
                for (int i = tid; i < V; i += THREADS) {   // a2: Philox counter (site, start lo, start hi, 0)
                    const u32x4 r = philox((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 0u, (uint32_t)P.seed,
                                           (uint32_t)(P.seed >> 32));
                    double sn, cs;
                    sincospi(unit_interval_pm1(r.x, r.y), &sn, &cs);
                    int pi, ri;
                    locate<N>(i, pi, ri);
                    (pi ? O : E)[(size_t)ri * 32 + L] = make_double2(cs, sn);
                }
#ifdef U1GF_TMA_PROF
                if (blockIdx.x == 0 && tid == 0) atomicAdd(&g_prof[5], (unsigned long long)(clock64() - prof_r0));
#endif
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
#ifdef U1GF_TMA_PROF
        if (blockIdx.x == 0 && tid == 0) atomicAdd(&g_prof[3], (unsigned long long)(clock64() - prof_s0));
#endif
        if (__ballot_sync(FULL, active) == 0) break;   // every warp holds the same lane states

        // ---------------------------------------------------------- odd half-sweep (second half of sweep t+1)
        {
            const bool commit = active && !fresh;
            fence_proxy_async();
            __syncthreads();
            PROF_T0();
            double unusedF = 0.0;
            accO = half_sweep<N, 1, W1>(S, O, O, nullptr, E, P.lnk + (size_t)HALF * 8, hs, warp, lane, P.k2, commit, false, skipped, unusedF);
            if (warp == 0) { PROF_ADD(2); }
            hs = (hs + 1) % G::HSMOD;   // the mbarrier phases only need hs modulo a multiple of 2 RW and 2 ST
            if (commit) ++t;
            fresh = false;
        }
        // ---------------------------------------------------------- even half-sweep (first half of sweep t+1)
        // lanes that can stop at this sweep (necessary conditions, known before the half-sweep): they save their even values
        if (warp < CW) sredO[warp * 32 + lane] = accO;
        fence_proxy_async();
        __syncthreads();
        double sumO = 0.0;   // odd part of the gauge precision of the field after sweep t, fixed order
#pragma unroll
        for (int w = 0; w < CW; ++w) sumO += sredO[w * 32 + lane];
        const bool cand = active && t > 0 && ((t % P.check_every == 0 && sumO / (double)V < P.eps) || t == P.max_sweeps);
        double accF = 0.0;
        const double accE = half_sweep<N, 0, W1>(S, E, E, SV, O, P.lnk, hs, warp, lane, P.k2, active, cand, skipped, accF);
        hs = (hs + 1) % G::HSMOD;
        // a4: gauge precision of the field after sweep t (R5), a5: F of that field; fixed summation order over the warps
        if (warp < CW) {
            sred[(rb * CW + warp) * 32 + lane] = accE;
            sredF[(rb * CW + warp) * 32 + lane] = accF;
        }
        __syncthreads();
        double Ssum = sumO, Fsum = 0.0;
#pragma unroll
        for (int w = 0; w < CW; ++w) {
            Ssum += sred[(rb * CW + w) * 32 + lane];
            Fsum += sredF[(rb * CW + w) * 32 + lane];
        }
        rb ^= 1;
        const bool conv = active && t > 0 && (t % P.check_every == 0) && (Ssum / (double)V < P.eps);
        maxed = active && !conv && t == P.max_sweeps;
        dumpm = __ballot_sync(FULL, conv || maxed);
        need = dumpm;
        if (warp == 0 && (conv || maxed)) s_F[lane] = Fsum;   // read by thread 0 behind the barriers of the finalisation
    }
#ifdef U1GF_TMA_PROF
    __syncthreads();
    if (blockIdx.x == 0 && tid == 0)
        printf("prof N=%d: producer waits on empty %llu, warp 0 waits on full %llu, odd half-sweeps (warp 0) %llu, service %llu cycles "
               "(finalisation loop of thread 0 %llu, refill loop %llu)\n", N, g_prof[0], g_prof[1], g_prof[2], g_prof[3], g_prof[4], g_prof[5]);
#endif
}

template <int N>
void fill_links(const u1gf_orbit* o, double2* dst) {
    using G = TG<N>;
    const double* U = o->U_host.data();
    for (int p = 0; p < 2; ++p)
        for (int g = 0; g < G::NS; ++g)
            for (int q = 0; q < G::SITES; ++q) {
                const int x3 = g / N, x2 = g % N, x1 = q / G::H, k = q % G::H;
                const int x0 = 2 * k + ((p + x1 + x2 + x3) & 1);
                const int x[4] = {x0, x1, x2, x3};
                const int i = x0 + N * (x1 + N * (x2 + N * x3));
                double2* e = dst + ((size_t)p * G::HALF + (size_t)g * G::SITES + q) * 8;
                int stride = 1;
                for (int mu = 0; mu < 4; ++mu) {
                    const int ib = i + (((x[mu] + N - 1) % N) - x[mu]) * stride;   // i - mu, periodic
                    e[mu] = make_double2(U[2 * (i * 4 + mu)], U[2 * (i * 4 + mu) + 1]);
                    e[4 + mu] = make_double2(U[2 * (ib * 4 + mu)], U[2 * (ib * 4 + mu) + 1]);
                    stride *= N;
                }
            }
}

template <int N, bool W1>
int launch_k(const u1gf_orbit* o, const RelaxArgs& a, TmaParams& P, cudaStream_t st) {
    using G = TG<N>;
    auto kern = relax_tma_kernel<N, W1>;
    U1GF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_bytes));
    unsigned long long teams = (unsigned long long)o->sm_count;   // one team per SM (shared memory)
    const unsigned long long batches = (a.n_starts + 31) / 32;
    if (teams > batches) teams = batches;
    // counter and team buffers start from zero (an idle lane then reads a null field, not stale bits)
    const size_t bytes = 256 + (size_t)teams * 3 * G::HALF * 32 * sizeof(double2);
    U1GF_CUDA(cudaMemsetAsync(a.workspace, 0, bytes, st));
    kern<<<(unsigned)teams, G::THREADS, G::smem_bytes, st>>>(P);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    return U1GF_OK;
}

template <int N>
int launch(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st) {
    const bool w1 = a.omega == 1.0;
    TmaParams P;
    P.seed = a.seed; P.first_start = a.first_start; P.n_starts = a.n_starts; P.start_ids = a.start_ids;
    P.k2 = w1 ? 0.0 : a.omega / (1.0 - a.omega); P.eps = a.eps;
    P.max_sweeps = a.max_sweeps; P.check_every = a.check_every;
    P.F_norm = a.F_norm; P.sweeps = a.sweeps; P.status = a.status; P.sig = a.sig; P.g_canon = a.g_canon;
    P.counter = (unsigned long long*)a.workspace;
    P.team_buf = (double2*)((char*)a.workspace + 256);
    P.lnk = o->U_tma;
    P.D = o->dev;
    return w1 ? launch_k<N, true>(o, a, P, st) : launch_k<N, false>(o, a, P, st);
}

int cubic4(int d, const int* ext) {
    if (d != 4 || ext[0] != ext[1] || ext[0] != ext[2] || ext[0] != ext[3]) return 0;
    return ext[0] == 6 || ext[0] == 8 ? ext[0] : 0;
}

}  // namespace

size_t tma_links_bytes(int d, const int* ext) { return cubic4(d, ext) ? (size_t)ext[0] * ext[0] * ext[0] * ext[0] * 8 * sizeof(double2) : 0; }

void tma_fill_links(const u1gf_orbit* o, double2* dst) {
    if (cubic4(o->dev.d, o->dev.ext) == 6) fill_links<6>(o, dst);
    else if (cubic4(o->dev.d, o->dev.ext) == 8) fill_links<8>(o, dst);
}

bool tma_supported(const u1gf_orbit* o) { return o->U_tma != nullptr && cubic4(o->dev.d, o->dev.ext) != 0; }

size_t tma_workspace_bytes(const u1gf_orbit* o, uint64_t n) {
    unsigned long long teams = (unsigned long long)o->sm_count;
    const unsigned long long batches = (n + 31) / 32;
    if (teams > batches) teams = batches;
    if (teams < 1) teams = 1;
    return 256 + (size_t)teams * 3 * (size_t)(o->dev.V / 2) * 32 * sizeof(double2);
}

int tma_relax(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st) {
    return cubic4(o->dev.d, o->dev.ext) == 6 ? launch<6>(o, a, st) : launch<8>(o, a, st);
}

}  // namespace u1gf
