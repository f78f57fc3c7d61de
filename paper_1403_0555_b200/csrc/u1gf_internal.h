// u1gf_internal.h -- shared declarations of the CUDA path (libu1gf.so).  Not part of the public ABI.
// Shares nothing with oracle/ (the CPU oracle is test infrastructure and carries its own generator).
#pragma once

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <vector>

#include "../../include/u1gf.h"

namespace u1gf {

// ------------------------------------------------------------------------------------------------------
// error plumbing
// ------------------------------------------------------------------------------------------------------
void set_error(const char* fmt, ...);
int fail(int code, const char* fmt, ...);
int check_device();  // U1GF_OK or U1GF_ENODEV (cached per thread)

#define U1GF_CUDA(call)                                                                        \
    do {                                                                                       \
        cudaError_t e__ = (call);                                                              \
        if (e__ != cudaSuccess)                                                                \
            return ::u1gf::fail(U1GF_ECUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e__), \
                                __FILE__, __LINE__);                                           \
    } while (0)

extern thread_local int t_launches;     // kernels of this library launched by the current call (CUB's not counted)

// ------------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11; the generator named at PAPER.md:L121, ref [59]).
// Own restatement of the published round function for the CUDA path, host + device.
// ------------------------------------------------------------------------------------------------------
struct u32x4 {
    uint32_t x, y, z, w;
};

__host__ __device__ __forceinline__ void mulhilo(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo) {
#ifdef __CUDA_ARCH__
    hi = __umulhi(a, b);
    lo = a * b;
#else
    const uint64_t p = (uint64_t)a * (uint64_t)b;
    hi = (uint32_t)(p >> 32);
    lo = (uint32_t)p;
#endif
}

__host__ __device__ __forceinline__ u32x4 philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                                 uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0, l0, h1, l1;
        mulhilo(0xD2511F53u, c0, h0, l0);
        mulhilo(0xCD9E8D57u, c2, h1, l1);
        const uint32_t a = h1 ^ c1 ^ k0;
        const uint32_t b = h0 ^ c3 ^ k1;
        c0 = a;
        c1 = l1;
        c2 = b;
        c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return u32x4{c0, c1, c2, c3};
}

// phase angle fraction v = 2u-1 in [-1,1), u = 53-bit uniform from words (lo, hi)
__host__ __device__ __forceinline__ double unit_interval_pm1(uint32_t lo, uint32_t hi) {
    const uint64_t r = (((uint64_t)hi << 32) | (uint64_t)lo) >> 11;
    return 2.0 * ((double)r * 1.1102230246251565e-16) - 1.0;  // exact: r*2^-53 is exact, 2u-1 exact
}

// ------------------------------------------------------------------------------------------------------
// orbit handle
// ------------------------------------------------------------------------------------------------------
constexpr int kMaxV = 8192;
constexpr int kMaxPhases = 10;  // 2 parities x (d'+1) levels, d' <= 4 odd extents

struct OrbitDev {
    int d, V;
    int ext[4];
    int n_phases;
    int phase_off[kMaxPhases + 1];  // phase p = order[phase_off[p] .. phase_off[p+1])
    int max_phase;                  // largest phase size
    int all_even;                   // every extent even: two phases, each link has one end in each
    const double2* U;               // [V*d] links, index i*d+mu
    const int* fwd;                 // [V*d] index of i+mu
    const int* bwd;                 // [V*d] index of i-mu
    const int* order;               // [V] sites sorted by (phase, index)
    const uint8_t* sgn;             // [V] signature sign bits: bit k = a_{k,i} is +1, bit 4+k = b_{k,i} is +1
    const uint8_t* fin;             // [V] 1: every neighbour of the site is updated before it in a sweep, so its Delta right
                                    //     after its own update is its Delta on the field after the sweep (phased kernel, R5)
};

}  // namespace u1gf

struct u1gf_orbit {
    u1gf::OrbitDev dev;          // device pointers + geometry (passed to kernels by value)
    std::vector<double> U_host;  // [V*d*2]
    void* blob = nullptr;        // one device allocation holding every table
    size_t blob_bytes = 0;
    int device = 0;
    int sm_count = 0;
    int kernel_choice = 0;  // 0 auto, 1 generic, 2 streamed with plain loads, 3 TMA-staged streamed (2, 3 fall back to generic where they do not apply)
    // device copy of the links in the layout of the specialised resident kernels (inside blob), or null
    const double2* U_lanes = nullptr;
    std::vector<double2> U_lanes_host;  // host copy of the links part of that table (kernel parameter of the NB == 1 kernels)
    // device copy of the links in the row order of the TMA-staged streamed kernel (inside blob), or null
    const double2* U_tma = nullptr;
    // u1gf_pipeline_host's memory of its last call on this handle: 1 = most starts were their own copy (n_distinct > n/4),
    // so the next call lets the first pass write the fields of all starts instead of relaxing the representatives again
    mutable int pipeline_keep_fields = 0;
};

namespace u1gf {

// relaxation back ends (relax_generic.cu, relax_lanes.cu)
struct RelaxArgs {
    uint64_t seed, first_start, n_starts;
    const uint64_t* start_ids;
    double omega, eps;
    int max_sweeps, check_every;
    double* F_norm;
    int32_t* sweeps;
    uint8_t* status;
    double* sig;
    double* g_canon;
    void* workspace;
    size_t workspace_bytes;
};

size_t generic_workspace_bytes(const u1gf_orbit* o, uint64_t n);
int generic_relax(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st);
// count_copies.cu: the de-duplication of all orbits of an ensemble in one pass (ensemble.cu picks it when the workspace allows)
size_t count_ens_onepass_workspace_bytes(unsigned n_orbits, uint64_t n_per);
int count_copies_ens_onepass(unsigned n_orbits, unsigned n_per, const double* F_norm, const double* sig, const uint8_t* status,
                             double tol_F, double tol_sig, int32_t* copy_id, int64_t* n_distinct, int64_t* rep,
                             int64_t* multiplicity, int64_t* hist, int nbins, void* workspace, cudaStream_t st);
// ensemble mode of the same kernel: n_orbits orbits of o's shape, links [n_orbits][V*d] at U_all, a.n_starts starts each
int generic_relax_ens(const u1gf_orbit* o, const double2* U_all, const unsigned long long* seeds, unsigned n_orbits,
                      const RelaxArgs& a, cudaStream_t st);
// redo mode: relax the starts at output positions pos[0 .. *n_dev) again (R6 fix-up of the resident kernels); `counter` is a
// zeroed device word
int generic_relax_list(const u1gf_orbit* o, const RelaxArgs& a, const unsigned* n_dev, const unsigned long long* pos,
                       unsigned long long* counter, cudaStream_t st);

// specialised "lane per start" resident kernels; lanes_supported() says whether the extents have one
bool lanes_supported(const u1gf_orbit* o);
const char* lanes_name(const u1gf_orbit* o);
size_t lanes_links_bytes(int d, const int* ext);  // extra blob bytes for the kernel's link layout (0 if none)
void lanes_fill_links(int d, const int* ext, const double* U_host, double2* dst_host);
size_t lanes_workspace_bytes(const u1gf_orbit* o, uint64_t n);
int lanes_relax(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st);
// ensemble mode: n_orbits orbits of the shape of `o` in one launch; U_all = their lanes tables, lanes_stride
// double2 apart; seeds_dev[n_orbits]; a.n_starts = starts per orbit; outputs at orbit * a.n_starts + k; a.start_ids unused
size_t lanes_ens_workspace_bytes(const u1gf_orbit* o, unsigned n_orbits, uint64_t n);
int lanes_relax_ens(const u1gf_orbit* o, const double2* U_all, unsigned long long lanes_stride,
                    const unsigned long long* seeds_dev, unsigned n_orbits, const RelaxArgs& a, cudaStream_t st);

// streamed "lane per start" kernel for the large even lattices (relax_stream.cu)
bool stream_supported(const u1gf_orbit* o);   // every extent even
bool stream_preferred(const u1gf_orbit* o);   // ... and large enough to be the automatic choice
size_t stream_workspace_bytes(const u1gf_orbit* o, uint64_t n);
int stream_relax(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st);

// TMA-staged streamed kernel for 6^4 and 8^4 (relax_tma.cu)
size_t tma_links_bytes(int d, const int* ext);   // extra blob bytes for its link table (0 if the extents have no such kernel)
void tma_fill_links(const u1gf_orbit* o, double2* dst_host);
bool tma_supported(const u1gf_orbit* o);
size_t tma_workspace_bytes(const u1gf_orbit* o, uint64_t n);
int tma_relax(const u1gf_orbit* o, const RelaxArgs& a, cudaStream_t st);

}  // namespace u1gf
