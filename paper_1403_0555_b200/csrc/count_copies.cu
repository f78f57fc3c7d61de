// count_copies.cu -- a8 de-duplication and counting of converged starts.
// The paper sorts the functional values on the GPU (bitonic sort) and counts distinct ones at 1e-8 resolution
// (PAPER.md:L129-135, L149).  Here: radix sort on the order-preserving integer image of F/(dV), maximal runs of
// gaps <= tol_F, leader election inside runs with the signature test (R7, R8), discovery-order numbering (L149),
// multiplicities and the histogram of PAPER.md:L167 (R15).  All integer work; no floating-point atomics.
#include <cooperative_groups.h>

#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include "u1gf_internal.h"

namespace cg = cooperative_groups;

namespace u1gf {
namespace {

constexpr unsigned kNone = 0xffffffffu;

struct Work {
    unsigned long long* keys_in;
    unsigned long long* keys_out;
    unsigned* pos_in;
    unsigned* pos_out;   // sorted order: pos_out[j] = position of the j-th smallest F
    unsigned* run_id;    // [n] flags, then inclusive scan - 1
    unsigned* run_min0;  // [n] leader candidate per run (two buffers alternate between rounds)
    unsigned* run_min1;
    int* leader_of;      // [n] by position
    unsigned* lead_idx;  // [n] is-leader flags, then exclusive scan = copy id of a leader
    unsigned* small;     // [0] n_conv, [1..2] remaining flags
    void* cub_tmp;
    size_t cub_bytes;
};

size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

size_t cub_temp_bytes(size_t n) {
    size_t a = 0, b = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, a, (unsigned long long*)nullptr, (unsigned long long*)nullptr,
                                    (unsigned*)nullptr, (unsigned*)nullptr, (int)n);
    cub::DeviceScan::InclusiveSum(nullptr, b, (unsigned*)nullptr, (unsigned*)nullptr, (int)n);
    size_t c = 0;   // the ensemble path's second, stable pass over 32-bit orbit indices
    cub::DeviceRadixSort::SortPairs(nullptr, c, (unsigned*)nullptr, (unsigned*)nullptr, (unsigned*)nullptr, (unsigned*)nullptr, (int)n);
    a = a > c ? a : c;
    return a > b ? a : b;
}

size_t carve(Work& w, size_t n, char* base) {
    size_t off = 0;
    auto take = [&](size_t bytes) {
        char* p = base ? base + off : nullptr;
        off += align256(bytes);
        return p;
    };
    const size_t m = n ? n : 1;
    w.keys_in = (unsigned long long*)take(m * 8);
    w.keys_out = (unsigned long long*)take(m * 8);
    w.pos_in = (unsigned*)take(m * 4);
    w.pos_out = (unsigned*)take(m * 4);
    w.run_id = (unsigned*)take(m * 4);
    w.run_min0 = (unsigned*)take(m * 4);
    w.run_min1 = (unsigned*)take(m * 4);
    w.leader_of = (int*)take(m * 4);
    w.lead_idx = (unsigned*)take(m * 4);
    w.small = (unsigned*)take(64);
    w.cub_bytes = cub_temp_bytes(m);
    w.cub_tmp = take(w.cub_bytes);
    return off;
}

// order-preserving map double -> uint64; records that did not converge sort to the very end
__global__ void make_keys_kernel(unsigned n, const double* __restrict__ F, const uint8_t* __restrict__ status, Work w,
                                 int64_t* multiplicity, int64_t* hist, int nbins) {
    const unsigned stride = gridDim.x * blockDim.x;
    unsigned local = 0;
    for (unsigned p = blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        unsigned long long key = ~0ull;
        if (!(status[p] & 1)) {
            const unsigned long long b = (unsigned long long)__double_as_longlong(F[p]);
            key = (b >> 63) ? ~b : (b | 0x8000000000000000ull);
            ++local;
        }
        w.keys_in[p] = key;
        w.pos_in[p] = p;
        w.leader_of[p] = -1;
        w.run_min0[p] = kNone;
        w.run_min1[p] = kNone;
        multiplicity[p] = 0;
    }
    if (hist)
        for (unsigned b = blockIdx.x * blockDim.x + threadIdx.x; b < (unsigned)nbins; b += stride) hist[b] = 0;
    local = __reduce_add_sync(0xffffffffu, local);
    if ((threadIdx.x & 31) == 0 && local) atomicAdd(&w.small[0], local);
}

// run heads: gap to the predecessor in sorted order exceeds tol_F
__global__ void run_flags_kernel(unsigned n, const double* __restrict__ F, double tol_F, Work w) {
    const unsigned n_conv = w.small[0];
    const unsigned stride = gridDim.x * blockDim.x;
    for (unsigned j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        unsigned f = 0;
        if (j < n_conv) f = (j == 0) ? 1u : ((F[w.pos_out[j]] - F[w.pos_out[j - 1]] > tol_F) ? 1u : 0u);
        w.run_id[j] = f;
    }
}

// leader election inside runs, repeated until every converged record has a leader
__global__ void __launch_bounds__(256) elect_kernel(const double* __restrict__ sig, double tol_sig, Work w) {
    cg::grid_group grid = cg::this_grid();
    const unsigned n_conv = w.small[0];
    const unsigned stride = gridDim.x * blockDim.x, t0 = blockIdx.x * blockDim.x + threadIdx.x;
    const double4* S = reinterpret_cast<const double4*>(sig);
    volatile unsigned* rem = w.small + 1;
    for (unsigned round = 0;; ++round) {
        unsigned* cur = (round & 1) ? w.run_min1 : w.run_min0;
        unsigned* nxt = (round & 1) ? w.run_min0 : w.run_min1;
        if (t0 == 0) rem[(round + 1) & 1] = 0;
        // candidates: the smallest position among the unassigned records of each run.  Sorted order puts the records of a
        // run next to each other, so the lanes of a warp mostly share a run: one atomic per run and warp (2^22 starts
        // in 5 copies would otherwise send 4 million atomics to 5 addresses)
        for (unsigned jb = t0 - (threadIdx.x & 31); jb < n_conv; jb += stride) {   // warp-uniform trip count
            const unsigned j = jb + (threadIdx.x & 31);
            unsigned r = kNone, p = kNone;
            if (j < n_conv) {
                p = w.pos_out[j];
                if (w.leader_of[p] < 0) r = w.run_id[j] - 1;
            }
            const unsigned peers = __match_any_sync(0xffffffffu, r);
            const unsigned pmin = __reduce_min_sync(peers, p);
            if (r != kNone && (threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1)) atomicMin(&cur[r], pmin);
        }
        grid.sync();
        bool left = false;
        for (unsigned j = t0; j < n_conv; j += stride) {
            const unsigned p = w.pos_out[j];
            if (w.leader_of[p] >= 0) continue;
            const unsigned r = w.run_id[j] - 1;
            const unsigned lead = __ldcg(&cur[r]);
            const double4 a = S[p], b = S[lead];
            const double dist = fmax(fmax(fabs(a.x - b.x), fabs(a.y - b.y)), fmax(fabs(a.z - b.z), fabs(a.w - b.w)));
            if (dist <= tol_sig) {
                w.leader_of[p] = (int)lead;
            } else {
                left = true;
                nxt[r] = kNone;  // was used two rounds ago; nobody reads it in this round
            }
        }
        if (__syncthreads_or(left ? 1 : 0) && threadIdx.x == 0) rem[(round + 1) & 1] = 1;
        grid.sync();
        if (!rem[(round + 1) & 1]) break;
    }
    const unsigned n_all = w.small[3];  // all records
    for (unsigned p = t0; p < n_all; p += stride) w.lead_idx[p] = (__ldcg(&w.leader_of[p]) == (int)p) ? 1u : 0u;
}

__global__ void assign_kernel(unsigned n, Work w, int32_t* copy_id, int64_t* n_distinct, int64_t* rep,
                              int64_t* multiplicity) {
    const unsigned stride = gridDim.x * blockDim.x;
    const unsigned nb = (n + 31) / 32 * 32;
    for (unsigned p = blockIdx.x * blockDim.x + threadIdx.x; p < nb; p += stride) {
        int id = -1;
        if (p < n) {
            const int lead = w.leader_of[p];
            if (lead >= 0) id = (int)w.lead_idx[lead];
            copy_id[p] = id;
            if (lead == (int)p) rep[id] = (int64_t)p;
            if (p == n - 1) *n_distinct = (int64_t)w.lead_idx[p] + (lead == (int)p ? 1 : 0);
        }
        // warp-aggregated integer atomics: one add per distinct id in the warp
        const unsigned peers = __match_any_sync(0xffffffffu, id);
        if (id >= 0 && (threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1))
            atomicAdd((unsigned long long*)&multiplicity[id], (unsigned long long)__popc(peers));
    }
}

__global__ void hist_kernel(const double* __restrict__ F, const int64_t* n_distinct, const int64_t* rep,
                            const int64_t* multiplicity, int64_t* hist, int nbins) {
    const int64_t nd = *n_distinct;
    for (int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; c < nd; c += (int64_t)gridDim.x * blockDim.x) {
        long long b = (long long)floor(F[rep[c]] * (double)nbins);
        b = b < 0 ? 0 : (b > nbins - 1 ? nbins - 1 : b);
        atomicAdd((unsigned long long*)&hist[b], (unsigned long long)multiplicity[c]);
    }
}

// ---- one pass over a whole ensemble: positions p = orbit * n_per + local position; the records are sorted by F and then,
// stably, by orbit index, so that every orbit's converged records lie together in F order and the records that did not
// converge (orbit key n_orbits) come last; a run never crosses an orbit boundary; leaders, and with them the global copy
// ids, come out orbit by orbit, and the id inside the orbit is the global id minus the number of leaders before the orbit.
__global__ void orbit_keys_kernel(unsigned n, unsigned n_per, unsigned n_orbits, const unsigned long long* __restrict__ keys_sorted,
                                  const unsigned* __restrict__ pos_sorted, unsigned* __restrict__ okeys) {
    const unsigned stride = gridDim.x * blockDim.x;
    for (unsigned j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride)
        okeys[j] = keys_sorted[j] == ~0ull ? n_orbits : pos_sorted[j] / n_per;
}

__global__ void run_flags_ens_kernel(unsigned n, unsigned n_per, const double* __restrict__ F, double tol_F, Work w) {
    const unsigned n_conv = w.small[0];
    const unsigned stride = gridDim.x * blockDim.x;
    for (unsigned j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        unsigned f = 0;
        if (j < n_conv) {
            const unsigned p = w.pos_out[j], q = j ? w.pos_out[j - 1] : 0u;
            f = (j == 0 || p / n_per != q / n_per) ? 1u : ((F[p] - F[q] > tol_F) ? 1u : 0u);
        }
        w.run_id[j] = f;
    }
}

__global__ void assign_ens_kernel(unsigned n, unsigned n_per, Work w, int32_t* copy_id, int64_t* n_distinct, int64_t* rep,
                                  int64_t* multiplicity) {
    const unsigned stride = gridDim.x * blockDim.x;
    const unsigned nb = (n + 31) / 32 * 32;
    for (unsigned p = blockIdx.x * blockDim.x + threadIdx.x; p < nb; p += stride) {
        int gid = -1;
        unsigned long long slot = 0;
        if (p < n) {
            const unsigned o = p / n_per, first = o * n_per;
            const unsigned base = w.lead_idx[first];   // leaders before this orbit (exclusive scan at its first position)
            const int lead = w.leader_of[p];
            int id = -1;
            if (lead >= 0) {
                gid = (int)w.lead_idx[lead];
                id = gid - (int)base;
                slot = (unsigned long long)first + (unsigned)id;
            }
            copy_id[p] = id;
            if (lead == (int)p) rep[slot] = (int64_t)(p - first);
            if (p == first + n_per - 1) n_distinct[o] = (int64_t)w.lead_idx[p] + (lead == (int)p ? 1 : 0) - (int64_t)base;
        }
        const unsigned peers = __match_any_sync(0xffffffffu, gid);
        if (gid >= 0 && (threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1))
            atomicAdd((unsigned long long*)&multiplicity[slot], (unsigned long long)__popc(peers));
    }
}

__global__ void hist_ens_kernel(unsigned n, unsigned n_per, const double* __restrict__ F, const int64_t* __restrict__ n_distinct,
                                const int64_t* __restrict__ rep, const int64_t* __restrict__ multiplicity, int64_t* hist, int nbins) {
    const unsigned stride = gridDim.x * blockDim.x;
    for (unsigned p = blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        const unsigned o = p / n_per, c = p - o * n_per;
        if ((int64_t)c >= n_distinct[o]) continue;
        long long b = (long long)floor(F[(size_t)o * n_per + (size_t)rep[p]] * (double)nbins);
        b = b < 0 ? 0 : (b > nbins - 1 ? nbins - 1 : b);
        atomicAdd((unsigned long long*)&hist[(size_t)o * nbins + b], (unsigned long long)multiplicity[p]);
    }
}

__global__ void init_small_kernel(unsigned* small, unsigned n) {
    if (threadIdx.x == 0) {
        small[0] = 0u;
        small[1] = 1u;
        small[2] = 0u;
        small[3] = n;
    }
}

__global__ void empty_kernel(int64_t* n_distinct, int64_t* hist, int nbins) {
    if (threadIdx.x == 0 && blockIdx.x == 0) *n_distinct = 0;
    if (hist)
        for (int b = threadIdx.x; b < nbins; b += blockDim.x) hist[b] = 0;
}

}  // namespace

size_t count_ens_onepass_workspace_bytes(unsigned n_orbits, uint64_t n_per) {
    const unsigned long long n = (unsigned long long)n_orbits * n_per;
    if (n == 0 || n >= (1ull << 31)) return 0;
    Work w;
    return carve(w, (size_t)n, nullptr);
}

// u1gf_count_copies for all orbits of an ensemble at once (same outputs as the per-orbit loop of ensemble.cu).
int count_copies_ens_onepass(unsigned n_orbits, unsigned n_per, const double* F_norm, const double* sig, const uint8_t* status,
                             double tol_F, double tol_sig, int32_t* copy_id, int64_t* n_distinct, int64_t* rep,
                             int64_t* multiplicity, int64_t* hist, int nbins, void* workspace, cudaStream_t st) {
    const unsigned n = n_orbits * n_per;
    Work w;
    carve(w, n, (char*)workspace);
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const unsigned blocks = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)sms * 8);
    int launches = 0;
    init_small_kernel<<<1, 32, 0, st>>>(w.small, n);
    U1GF_CUDA(cudaGetLastError());
    make_keys_kernel<<<blocks, 256, 0, st>>>(n, F_norm, status, w, multiplicity, hist, hist ? (int)n_orbits * nbins : 0);
    U1GF_CUDA(cudaGetLastError());
    launches += 2;
    size_t tb = w.cub_bytes;
    U1GF_CUDA(cub::DeviceRadixSort::SortPairs(w.cub_tmp, tb, w.keys_in, w.keys_out, w.pos_in, w.pos_out, (int)n, 0, 64, st));
    // second, stable pass: orbit index as the major key.  The 64-bit input keys are no longer needed: their array holds
    // the two 32-bit key arrays of this pass; the positions go back into pos_in, which becomes the sorted order
    unsigned* ok_in = (unsigned*)w.keys_in;
    unsigned* ok_out = ok_in + n;
    orbit_keys_kernel<<<blocks, 256, 0, st>>>(n, n_per, n_orbits, w.keys_out, w.pos_out, ok_in);
    U1GF_CUDA(cudaGetLastError());
    ++launches;
    int bits = 1;
    while ((1u << bits) <= n_orbits) ++bits;
    tb = w.cub_bytes;
    U1GF_CUDA(cub::DeviceRadixSort::SortPairs(w.cub_tmp, tb, ok_in, ok_out, w.pos_out, w.pos_in, (int)n, 0, bits, st));
    std::swap(w.pos_in, w.pos_out);
    run_flags_ens_kernel<<<blocks, 256, 0, st>>>(n, n_per, F_norm, tol_F, w);
    U1GF_CUDA(cudaGetLastError());
    ++launches;
    tb = w.cub_bytes;
    U1GF_CUDA(cub::DeviceScan::InclusiveSum(w.cub_tmp, tb, w.run_id, w.run_id, (int)n, st));
    {
        int per_sm = 0;
        U1GF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, elect_kernel, 256, 0));
        unsigned grid = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)per_sm * sms);
        if (grid < 1) grid = 1;
        void* args[] = {(void*)&sig, (void*)&tol_sig, (void*)&w};
        U1GF_CUDA(cudaLaunchCooperativeKernel((void*)elect_kernel, dim3(grid), dim3(256), args, 0, st));
        ++launches;
    }
    tb = w.cub_bytes;
    U1GF_CUDA(cub::DeviceScan::ExclusiveSum(w.cub_tmp, tb, w.lead_idx, w.lead_idx, (int)n, st));
    assign_ens_kernel<<<blocks, 256, 0, st>>>(n, n_per, w, copy_id, n_distinct, rep, multiplicity);
    U1GF_CUDA(cudaGetLastError());
    ++launches;
    if (hist) {
        hist_ens_kernel<<<blocks, 256, 0, st>>>(n, n_per, F_norm, n_distinct, rep, multiplicity, hist, nbins);
        U1GF_CUDA(cudaGetLastError());
        ++launches;
    }
    t_launches = launches;
    return U1GF_OK;
}

}  // namespace u1gf

using namespace u1gf;

extern "C" {

size_t u1gf_count_workspace_bytes(uint64_t n) {
    if (n >= (1ull << 31)) return 0;
    Work w;
    return carve(w, (size_t)n, nullptr);
}

int u1gf_count_copies(uint64_t n_, const double* F_norm, const double* sig, const uint8_t* status, double tol_F,
                      double tol_sig, int32_t* copy_id, int64_t* n_distinct, int64_t* rep, int64_t* multiplicity,
                      int64_t* hist, int32_t nbins, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    t_launches = 0;
    if (n_ >= (1ull << 31)) return fail(U1GF_EINVAL, "u1gf_count_copies: n must be below 2^31");
    if (!n_distinct) return fail(U1GF_EINVAL, "u1gf_count_copies: NULL n_distinct");
    if (hist && nbins < 1) return fail(U1GF_EINVAL, "u1gf_count_copies: nbins must be >= 1 when hist is given");
    if (!(tol_F >= 0.0) || !(tol_sig >= 0.0)) return fail(U1GF_EINVAL, "u1gf_count_copies: negative tolerance");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned n = (unsigned)n_;
    if (n == 0) {
        empty_kernel<<<1, 256, 0, st>>>(n_distinct, hist, nbins);
        U1GF_CUDA(cudaGetLastError());
        ++t_launches;
        return U1GF_OK;
    }
    if (!F_norm || !sig || !status || !copy_id || !rep || !multiplicity)
        return fail(U1GF_EINVAL, "u1gf_count_copies: NULL array");
    Work w;
    const size_t need = carve(w, n, nullptr);
    if (!workspace || workspace_bytes < need)
        return fail(U1GF_ENOMEM, "u1gf_count_copies: workspace of %zu bytes needed, %zu given", need, workspace_bytes);
    if (((uintptr_t)workspace & 255) != 0) return fail(U1GF_EINVAL, "u1gf_count_copies: workspace not 256-byte aligned");
    carve(w, n, (char*)workspace);

    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const unsigned blocks = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)sms * 8);

    init_small_kernel<<<1, 32, 0, st>>>(w.small, n);   // on the device: no staged copy from pageable host memory
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    make_keys_kernel<<<blocks, 256, 0, st>>>(n, F_norm, status, w, multiplicity, hist, nbins);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    size_t tb = w.cub_bytes;
    U1GF_CUDA(cub::DeviceRadixSort::SortPairs(w.cub_tmp, tb, w.keys_in, w.keys_out, w.pos_in, w.pos_out, (int)n, 0, 64, st));
    run_flags_kernel<<<blocks, 256, 0, st>>>(n, F_norm, tol_F, w);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    tb = w.cub_bytes;
    U1GF_CUDA(cub::DeviceScan::InclusiveSum(w.cub_tmp, tb, w.run_id, w.run_id, (int)n, st));

    {
        int per_sm = 0;
        U1GF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, elect_kernel, 256, 0));
        unsigned grid = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)per_sm * sms);
        if (grid < 1) grid = 1;
        void* args[] = {(void*)&sig, (void*)&tol_sig, (void*)&w};
        U1GF_CUDA(cudaLaunchCooperativeKernel((void*)elect_kernel, dim3(grid), dim3(256), args, 0, st));
        ++t_launches;
    }
    tb = w.cub_bytes;
    U1GF_CUDA(cub::DeviceScan::ExclusiveSum(w.cub_tmp, tb, w.lead_idx, w.lead_idx, (int)n, st));
    // leader flags were overwritten by their scan; assign_kernel recognises leaders by leader_of[p] == p
    assign_kernel<<<blocks, 256, 0, st>>>(n, w, copy_id, n_distinct, rep, multiplicity);
    U1GF_CUDA(cudaGetLastError());
    ++t_launches;
    if (hist) {
        hist_kernel<<<blocks, 256, 0, st>>>(F_norm, n_distinct, rep, multiplicity, hist, nbins);
        U1GF_CUDA(cudaGetLastError());
        ++t_launches;
    }
    return U1GF_OK;
}

}  // extern "C"
