// u1gf_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, step-by-step CPU oracle (C++17, FP64, scalar loops) for the hot path of
// Mehta & Schroeck, "Enumerating Copies in the First Gribov Region on the Lattice in up to
// four Dimensions" (arXiv:1403.0555): compact-U(1) lattice-Landau-gauge relaxation from
// seeded random gauge transformations.  Citations are PAPER.md:L<line> plus the section /
// equation, and DESIGN.md "Readings" R<k> where the paper is silent.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this file's shared object.  It shares no code, header, table or constant generator with
// paper_1403_0555_b200/csrc (the CUDA path) and neither includes the other.
//
// Conventions (BASELINE naming, i.e. links theta, gauge angles phi):
//   site index   i = x0 + N0*(x1 + N1*(x2 + N2*x3)), periodic in every direction
//   link         U_{i,mu} = (cos theta_{i,mu}, sin theta_{i,mu})
//   gauge field  g_i = (cos phi_i, sin phi_i)
//   transformed  U^g_{i,mu} = g_i U_{i,mu} conj(g_{i+mu})                 (Eq. 5 convention, R1)
//   functional   F[g] = sum_{i,mu} Re(g_i U_{i,mu} conj(g_{i+mu}))        (Eq. 3, maximised; x = 1 - F/(dV))
//   all complex numbers are stored as interleaved (re, im) doubles.
//
// Pinned by tests/test_oracle_*.py (-m "not gpu"): angle-form cross-check, brute-force grid
// scans on 2x2 and 3x2, cold-orbit twist closed forms, pure-gauge orbit, gauge covariance,
// the 1-D ring closed form, per-sweep invariants, Philox known answers.  The start -> copy
// ASSIGNMENT for a given seed has no external pin ("parity unpinned" for that map only).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11 -- the generator the paper names, ref [59]
// L311).  Restated from the published algorithm: two 32x32->64 multiplies per round, ten rounds,
// Weyl key schedule.
// ---------------------------------------------------------------------------------------------
struct Philox4 { uint32_t v[4]; };

Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // round multipliers
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // Weyl increments (golden ratio, sqrt(3)-1)
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)M0 * c0;
        const uint64_t p1 = (uint64_t)M1 * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    return Philox4{{c0, c1, c2, c3}};
}

// 53-bit uniform in [0,1) from words (x0 low, x1 high)  (O2)
inline double u53(uint32_t x0, uint32_t x1) {
    const uint64_t r = (((uint64_t)x1 << 32) | (uint64_t)x0) >> 11;
    return (double)r * (1.0 / 9007199254740992.0);  // 2^-53
}

// ---------------------------------------------------------------------------------------------
// Lattice geometry: periodic neighbours, parity.
// ---------------------------------------------------------------------------------------------
struct Lattice {
    int d = 0;
    int ext[4] = {1, 1, 1, 1};
    int V = 0;
    std::vector<int> fwd;     // fwd[i*d+mu] = index of i + mu^
    std::vector<int> bwd;     // bwd[i*d+mu] = index of i - mu^
    std::vector<int> parity;  // (sum_mu x_mu) mod 2
};

bool make_lattice(int d, const int32_t* extents, Lattice& L) {
    if (d < 1 || d > 4 || extents == nullptr) return false;
    L.d = d;
    long V = 1;
    for (int mu = 0; mu < d; ++mu) {
        if (extents[mu] < 2) return false;
        L.ext[mu] = extents[mu];
        V *= extents[mu];
        if (V > (1 << 24)) return false;
    }
    L.V = (int)V;
    L.fwd.assign((size_t)L.V * d, 0);
    L.bwd.assign((size_t)L.V * d, 0);
    L.parity.assign(L.V, 0);
    for (int i = 0; i < L.V; ++i) {
        int x[4] = {0, 0, 0, 0};
        int r = i, s = 0;
        for (int mu = 0; mu < d; ++mu) { x[mu] = r % L.ext[mu]; r /= L.ext[mu]; s += x[mu]; }
        L.parity[i] = s & 1;
        int stride = 1;
        for (int mu = 0; mu < d; ++mu) {
            const int xp = (x[mu] + 1) % L.ext[mu];
            const int xm = (x[mu] + L.ext[mu] - 1) % L.ext[mu];
            L.fwd[(size_t)i * d + mu] = i + (xp - x[mu]) * stride;
            L.bwd[(size_t)i * d + mu] = i + (xm - x[mu]) * stride;
            stride *= L.ext[mu];
        }
    }
    return true;
}

// O1: U_{i,mu} = (cos theta, sin theta), libm
void make_links(const Lattice& L, const double* theta, std::vector<double>& U) {
    const size_t nl = (size_t)L.V * L.d;
    U.resize(2 * nl);
    for (size_t l = 0; l < nl; ++l) {
        U[2 * l] = std::cos(theta[l]);
        U[2 * l + 1] = std::sin(theta[l]);
    }
}

// w_i = sum_{mu=0}^{d-1} [ conj(U_{i,mu}) g_{i+mu} + U_{i-mu,mu} g_{i-mu} ]  ( = conj(K_i), Eq. 5, PAPER.md:L95 )
inline void neighbour_sum(const Lattice& L, const double* U, const double* g, int i, double& wr, double& wi) {
    wr = 0.0; wi = 0.0;
    for (int mu = 0; mu < L.d; ++mu) {
        const int jf = L.fwd[(size_t)i * L.d + mu];
        const int jb = L.bwd[(size_t)i * L.d + mu];
        const double ur = U[2 * ((size_t)i * L.d + mu)], ui = U[2 * ((size_t)i * L.d + mu) + 1];
        const double br = U[2 * ((size_t)jb * L.d + mu)], bi = U[2 * ((size_t)jb * L.d + mu) + 1];
        const double gfr = g[2 * jf], gfi = g[2 * jf + 1];
        const double gbr = g[2 * jb], gbi = g[2 * jb + 1];
        // conj(U) * g_fwd
        wr += ur * gfr + ui * gfi;
        wi += ur * gfi - ui * gfr;
        // U_back * g_bwd
        wr += br * gbr - bi * gbi;
        wi += br * gbi + bi * gbr;
    }
}

// O3: one full sweep = parity 0 then parity 1, sites in increasing index order, IN PLACE.
// For even extents this equals the paper's concurrent checkerboard update; for odd
// extents the sequential order is the definition (reading R3).  Local solution g_i <- w/|w|
// followed by the over-relaxation mix h = (1-omega) g + omega g^, g <- h/|h| (R2;
// omega = 1 is the paper's algorithm, which declines over-relaxation).
// Returns true if some site had |w|^2 < 1e-280 and was left unchanged (R6).
bool sweep_in_place(const Lattice& L, const double* U, double* g, double omega) {
    bool skipped = false;
    for (int p = 0; p < 2; ++p) {
        for (int i = 0; i < L.V; ++i) {
            if (L.parity[i] != p) continue;
            double wr, wi;
            neighbour_sum(L, U, g, i, wr, wi);
            const double n = wr * wr + wi * wi;
            if (n < 1e-280) { skipped = true; continue; }
            const double s = std::sqrt(n);
            const double ghr = wr / s, ghi = wi / s;
            const double hr = (1.0 - omega) * g[2 * i] + omega * ghr;
            const double hi = (1.0 - omega) * g[2 * i + 1] + omega * ghi;
            const double m = std::sqrt(hr * hr + hi * hi);
            g[2 * i] = hr / m;
            g[2 * i + 1] = hi / m;
        }
    }
    return skipped;
}

// O4: Delta_i = Im(g_i conj(w_i)) on the given field; vartheta = (1/V) sum_i Delta_i^2.
double gauge_precision(const Lattice& L, const double* U, const double* g, double* Delta /*[V] or null*/) {
    double acc = 0.0;
    for (int i = 0; i < L.V; ++i) {
        double wr, wi;
        neighbour_sum(L, U, g, i, wr, wi);
        const double D = g[2 * i + 1] * wr - g[2 * i] * wi;
        if (Delta) Delta[i] = D;
        acc += D * D;
    }
    return acc / (double)L.V;
}

// O5: F = sum_{i,mu} Re( g_i U_{i,mu} conj(g_{i+mu}) )   (Eq. 3, in the R1 convention)
double functional(const Lattice& L, const double* U, const double* g) {
    double F = 0.0;
    for (int i = 0; i < L.V; ++i) {
        for (int mu = 0; mu < L.d; ++mu) {
            const int j = L.fwd[(size_t)i * L.d + mu];
            const double ur = U[2 * ((size_t)i * L.d + mu)], ui = U[2 * ((size_t)i * L.d + mu) + 1];
            // a = g_i * U
            const double ar = g[2 * i] * ur - g[2 * i + 1] * ui;
            const double ai = g[2 * i] * ui + g[2 * i + 1] * ur;
            // Re(a * conj(g_j))
            F += ar * g[2 * j] + ai * g[2 * j + 1];
        }
    }
    return F;
}

// O2: random start s: g_i = (cos pi v, sin pi v), v = 2u-1, u 53-bit uniform from
// Philox key (seed_lo, seed_hi), counter (i, s_lo, s_hi, 0)
void make_start(int V, uint64_t seed, uint64_t s, double* g) {
    const double pi = 3.14159265358979323846;
    for (int i = 0; i < V; ++i) {
        const Philox4 r = philox4x32_10((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 0u,
                                        (uint32_t)seed, (uint32_t)(seed >> 32));
        const double u = u53(r.v[0], r.v[1]);
        const double v = 2.0 * u - 1.0;
        g[2 * i] = std::cos(pi * v);
        g[2 * i + 1] = std::sin(pi * v);
    }
}

// O6 signs: a_{k,i}, b_{k,i} in {+1,-1} from Philox key (0x51, 0), counter (i, k, 0, 1):
// a = +1 if bit 0 of word 0 is set else -1; b likewise from word 1.
inline void signature_signs(int i, int k, double& a, double& b) {
    const Philox4 r = philox4x32_10((uint32_t)i, (uint32_t)k, 0u, 1u, 0x51u, 0u);
    a = (r.v[0] & 1u) ? 1.0 : -1.0;
    b = (r.v[1] & 1u) ? 1.0 : -1.0;
}

// O6: g~_i = g_i conj(g_{V-1}) (angle at the last site (N,...,N) fixed to zero);
// signature p_k = (1/V) sum_i (a_{k,i} Re g~_i + b_{k,i} Im g~_i), k = 0..3.
void canonicalise(int V, const double* g, double* gc /*[2V]*/, double* sig /*[4]*/) {
    const double cr = g[2 * (V - 1)], ci = g[2 * (V - 1) + 1];
    for (int i = 0; i < V; ++i) {
        gc[2 * i] = g[2 * i] * cr + g[2 * i + 1] * ci;
        gc[2 * i + 1] = g[2 * i + 1] * cr - g[2 * i] * ci;
    }
    for (int k = 0; k < 4; ++k) {
        double acc = 0.0;
        for (int i = 0; i < V; ++i) {
            double a, b;
            signature_signs(i, k, a, b);
            acc += a * gc[2 * i] + b * gc[2 * i + 1];
        }
        sig[k] = acc / (double)V;
    }
}

}  // namespace

extern "C" {

// Raw generator, exposed for the known-answer pin (P10).
void u1gf_oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const Philox4 r = philox4x32_10(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1]);
    for (int k = 0; k < 4; ++k) out[k] = r.v[k];
}

// O1.  U_out[V*d*2].
int u1gf_oracle_links(int d, const int32_t* extents, const double* theta, double* U_out) {
    Lattice L;
    if (!make_lattice(d, extents, L)) return -1;
    std::vector<double> U;
    make_links(L, theta, U);
    std::memcpy(U_out, U.data(), U.size() * sizeof(double));
    return 0;
}

// O2.  g_out[V*2].
int u1gf_oracle_start(int V, uint64_t seed, uint64_t start, double* g_out) {
    if (V < 1) return -1;
    make_start(V, seed, start, g_out);
    return 0;
}

// O3 on a caller-supplied field (n_sweeps sweeps, in place); *skipped = 1 if an R6 skip occurred.
int u1gf_oracle_sweeps(int d, const int32_t* extents, const double* theta, double* g, double omega,
                       int32_t n_sweeps, int32_t* skipped) {
    Lattice L;
    if (!make_lattice(d, extents, L)) return -1;
    std::vector<double> U;
    make_links(L, theta, U);
    bool sk = false;
    for (int t = 0; t < n_sweeps; ++t) sk = sweep_in_place(L, U.data(), g, omega) || sk;
    if (skipped) *skipped = sk ? 1 : 0;
    return 0;
}

// O4 / O5 on a caller-supplied field.  Delta[V] may be null.
int u1gf_oracle_measure(int d, const int32_t* extents, const double* theta, const double* g,
                        double* F_out, double* vartheta_out, double* Delta) {
    Lattice L;
    if (!make_lattice(d, extents, L)) return -1;
    std::vector<double> U;
    make_links(L, theta, U);
    if (F_out) *F_out = functional(L, U.data(), g);
    if (vartheta_out) *vartheta_out = gauge_precision(L, U.data(), g, Delta);
    return 0;
}

// Neighbour sums w_i for every site (for the P8 pin F = 1/2 sum_i |w_i| at a stationary point).
int u1gf_oracle_neighbour_sums(int d, const int32_t* extents, const double* theta, const double* g, double* w /*[2V]*/) {
    Lattice L;
    if (!make_lattice(d, extents, L)) return -1;
    std::vector<double> U;
    make_links(L, theta, U);
    for (int i = 0; i < L.V; ++i) neighbour_sum(L, U.data(), g, i, w[2 * i], w[2 * i + 1]);
    return 0;
}

// O6 on a caller-supplied field.
int u1gf_oracle_canonicalise(int V, const double* g, double* g_canon, double* sig) {
    if (V < 1) return -1;
    canonicalise(V, g, g_canon, sig);
    return 0;
}

// Signature sign table (for inspection / tests): a[4*V], b[4*V] at index k*V+i.
int u1gf_oracle_signature_signs(int V, double* a, double* b) {
    for (int k = 0; k < 4; ++k)
        for (int i = 0; i < V; ++i) signature_signs(i, k, a[(size_t)k * V + i], b[(size_t)k * V + i]);
    return 0;
}

// O2-O6 for a batch of starts (the relaxation proper).  Start k uses index start_ids[k] if
// start_ids != null, else first_start + k.  Outputs per start k:
//   F_norm[k]   F/(dV) of the final field
//   sweeps[k]   number of full sweeps performed
//   status[k]   bit0: reached max_sweeps without passing the test; bit1: an R6 skip occurred
//   sig[4k..]   canonical signature
//   g_canon     [n*V*2] canonical field, or null
//   vt_stop[k]  vartheta at the last test performed (or -1 if none); vt_prev[k] the test before (or -1)
// Stop rule O4: after sweep t with t mod check_every == 0, vartheta_t < eps (PAPER.md:L133 in the
// per-start mean-square form of reading R5).
int u1gf_oracle_relax(int d, const int32_t* extents, const double* theta, uint64_t seed,
                      uint64_t first_start, uint64_t n_starts, const uint64_t* start_ids, double omega,
                      double eps, int32_t max_sweeps, int32_t check_every, double* F_norm, int32_t* sweeps,
                      uint8_t* status, double* sig, double* g_canon, double* vt_stop, double* vt_prev,
                      int32_t n_threads) {
    Lattice L;
    if (!make_lattice(d, extents, L)) return -1;
    if (!(omega >= 1.0 && omega < 2.0) || !(eps > 0.0) || max_sweeps < 1 || check_every < 1) return -1;
    std::vector<double> U;
    make_links(L, theta, U);
    const int V = L.V;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel
    {
        std::vector<double> g(2 * (size_t)V), gc(2 * (size_t)V);
#pragma omp for schedule(dynamic, 16)
        for (int64_t k = 0; k < (int64_t)n_starts; ++k) {
            const uint64_t s = start_ids ? start_ids[k] : first_start + (uint64_t)k;
            make_start(V, seed, s, g.data());
            uint8_t st = 1;  // not converged until a test passes
            bool skipped = false;
            int32_t t = 0;
            double vt = -1.0, vtp = -1.0;
            while (t < max_sweeps) {
                skipped = sweep_in_place(L, U.data(), g.data(), omega) || skipped;
                ++t;
                if (t % check_every == 0) {
                    vtp = vt;
                    vt = gauge_precision(L, U.data(), g.data(), nullptr);
                    if (vt < eps) { st = 0; break; }
                }
            }
            if (skipped) st |= 2;
            F_norm[k] = functional(L, U.data(), g.data()) / ((double)d * (double)V);
            sweeps[k] = t;
            status[k] = st;
            double sg[4];
            canonicalise(V, g.data(), gc.data(), sg);
            for (int q = 0; q < 4; ++q) sig[4 * k + q] = sg[q];
            if (g_canon) std::memcpy(g_canon + (size_t)k * 2 * V, gc.data(), 2 * (size_t)V * sizeof(double));
            if (vt_stop) vt_stop[k] = vt;
            if (vt_prev) vt_prev[k] = vtp;
        }
    }
    return 0;
}

// O7 (matrix part): dense Faddeev-Popov operator M[V*V] (row major) = Hessian of -F with respect to
// the gauge angles at g:  c_{i,mu} = Re(g_i U_{i,mu} conj(g_{i+mu}));
// (M v)_i = sum_mu [ c_{i,mu} (v_i - v_{i+mu}) + c_{i-mu,mu} (v_i - v_{i-mu}) ].
// Built link by link so that double bonds on extent-2 directions (R4) add up.
int u1gf_oracle_fp_matrix(int d, const int32_t* extents, const double* theta, const double* g, double* M) {
    Lattice L;
    if (!make_lattice(d, extents, L)) return -1;
    std::vector<double> U;
    make_links(L, theta, U);
    const size_t V = (size_t)L.V;
    std::memset(M, 0, V * V * sizeof(double));
    for (int i = 0; i < L.V; ++i) {
        for (int mu = 0; mu < L.d; ++mu) {
            const int j = L.fwd[(size_t)i * L.d + mu];
            const double ur = U[2 * ((size_t)i * L.d + mu)], ui = U[2 * ((size_t)i * L.d + mu) + 1];
            const double ar = g[2 * i] * ur - g[2 * i + 1] * ui;
            const double ai = g[2 * i] * ui + g[2 * i + 1] * ur;
            const double c = ar * g[2 * j] + ai * g[2 * j + 1];
            M[(size_t)i * V + i] += c;
            M[(size_t)j * V + j] += c;
            M[(size_t)i * V + j] -= c;
            M[(size_t)j * V + i] -= c;
        }
    }
    return 0;
}

int u1gf_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
