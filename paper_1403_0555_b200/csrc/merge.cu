// merge.cu -- SURVEY section 8(f)-4 / 8(e): merging the distinct-copy tables of several start ranges.
// The path shards over starts (the paper drives 4 GPUs from a host loop over independent samples); each
// shard de-duplicates its own starts (u1gf_count_copies) and ends with a table {F/(dV), signature, first start,
// multiplicity} per copy.  u1gf_merge_copy_tables applies the copy identity of reading R7 to the concatenated tables:
// the entries are put in order of their first start (the discovery order of the whole job), clustered
// exactly like starts are (sort by F, runs with gaps <= tol_F, leaders by first discovery, signature within tol_sig),
// and the merged copies are numbered by first discovery; multiplicities add up.
#include <cub/cub.cuh>

#include "u1gf_internal.h"

namespace u1gf {
namespace {

struct MergeWork {
    unsigned long long* key_in;   // first_start as sort key
    unsigned long long* key_out;
    unsigned* idx_in;             // entry index
    unsigned* perm;               // perm[j] = entry with the j-th smallest first_start
    double* F_s;                  // inputs of count_copies, in that order
    double* sig_s;
    uint8_t* status_s;
    int32_t* id_s;
    int64_t* rep_s;
    int64_t* mult_s;
    void* cub_tmp;
    size_t cub_bytes;
    void* count_ws;
    size_t count_bytes;
};

size_t carve(MergeWork& w, size_t m, char* base) {
    size_t off = 0;
    auto take = [&](size_t bytes) {
        char* p = base ? base + off : nullptr;
        off += (bytes + 255) & ~(size_t)255;
        return p;
    };
    const size_t mm = m ? m : 1;
    w.key_in = (unsigned long long*)take(mm * 8);
    w.key_out = (unsigned long long*)take(mm * 8);
    w.idx_in = (unsigned*)take(mm * 4);
    w.perm = (unsigned*)take(mm * 4);
    w.F_s = (double*)take(mm * 8);
    w.sig_s = (double*)take(mm * 32);
    w.status_s = (uint8_t*)take(mm);
    w.id_s = (int32_t*)take(mm * 4);
    w.rep_s = (int64_t*)take(mm * 8);
    w.mult_s = (int64_t*)take(mm * 8);
    size_t tb = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, tb, (unsigned long long*)nullptr, (unsigned long long*)nullptr,
                                    (unsigned*)nullptr, (unsigned*)nullptr, (int)mm);
    w.cub_bytes = tb;
    w.cub_tmp = take(tb);
    w.count_bytes = u1gf_count_workspace_bytes(mm);
    w.count_ws = take(w.count_bytes);
    return off;
}

__global__ void merge_keys_kernel(unsigned m, const int64_t* __restrict__ first_start, unsigned long long* key, unsigned* idx) {
    for (unsigned p = blockIdx.x * blockDim.x + threadIdx.x; p < m; p += gridDim.x * blockDim.x) {
        key[p] = (unsigned long long)first_start[p] ^ 0x8000000000000000ull;   // signed order
        idx[p] = p;
    }
}

__global__ void merge_gather_kernel(unsigned m, const unsigned* __restrict__ perm, const double* __restrict__ F,
                                    const double* __restrict__ sig, double* F_s, double* sig_s, uint8_t* status_s,
                                    int64_t* merged_multiplicity) {
    for (unsigned j = blockIdx.x * blockDim.x + threadIdx.x; j < m; j += gridDim.x * blockDim.x) {
        const unsigned e = perm[j];
        F_s[j] = F[e];
        reinterpret_cast<double4*>(sig_s)[j] = reinterpret_cast<const double4*>(sig)[e];
        status_s[j] = 0;
        merged_multiplicity[j] = 0;
    }
}

__global__ void merge_scatter_kernel(unsigned m, const unsigned* __restrict__ perm, const int32_t* __restrict__ id_s,
                                     const int64_t* __restrict__ rep_s, const int64_t* __restrict__ n_merged,
                                     const int64_t* __restrict__ first_start, const int64_t* __restrict__ multiplicity,
                                     int32_t* merged_id, int64_t* merged_first_start, int64_t* merged_multiplicity) {
    const int64_t nm = *n_merged;
    for (unsigned j = blockIdx.x * blockDim.x + threadIdx.x; j < m; j += gridDim.x * blockDim.x) {
        const unsigned e = perm[j];
        const int id = id_s[j];
        merged_id[e] = id;
        atomicAdd((unsigned long long*)&merged_multiplicity[id], (unsigned long long)multiplicity[e]);   // integer: order-free
        if ((int64_t)j < nm) merged_first_start[j] = first_start[perm[rep_s[j]]];
    }
}

}  // namespace
}  // namespace u1gf

using namespace u1gf;

extern "C" {

size_t u1gf_merge_workspace_bytes(uint64_t m) {
    if (m >= (1ull << 31)) return 0;
    MergeWork w;
    return carve(w, (size_t)m, nullptr);
}

int u1gf_merge_copy_tables(uint64_t m_, const double* F_rep, const double* sig_rep, const int64_t* first_start,
                           const int64_t* multiplicity, double tol_F, double tol_sig, int32_t* merged_id,
                           int64_t* n_merged, int64_t* merged_first_start, int64_t* merged_multiplicity,
                           void* workspace, size_t workspace_bytes, void* cuda_stream) {
    t_launches = 0;
    if (m_ >= (1ull << 31)) return fail(U1GF_EINVAL, "u1gf_merge_copy_tables: m must be below 2^31");
    if (!n_merged) return fail(U1GF_EINVAL, "u1gf_merge_copy_tables: NULL n_merged");
    if (int rc = check_device()) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (m_ == 0) {
        U1GF_CUDA(cudaMemsetAsync(n_merged, 0, sizeof(int64_t), st));
        return U1GF_OK;
    }
    if (!F_rep || !sig_rep || !first_start || !multiplicity || !merged_id || !merged_first_start || !merged_multiplicity)
        return fail(U1GF_EINVAL, "u1gf_merge_copy_tables: NULL array");
    MergeWork w;
    const size_t need = carve(w, (size_t)m_, nullptr);
    if (!workspace || workspace_bytes < need)
        return fail(U1GF_ENOMEM, "u1gf_merge_copy_tables: workspace of %zu bytes needed, %zu given", need, workspace_bytes);
    if (((uintptr_t)workspace & 255) != 0) return fail(U1GF_EINVAL, "u1gf_merge_copy_tables: workspace not 256-byte aligned");
    carve(w, (size_t)m_, (char*)workspace);
    const unsigned m = (unsigned)m_;
    const unsigned blocks = (m + 255) / 256 < 1184u ? (m + 255) / 256 : 1184u;
    int launches = 0;
    merge_keys_kernel<<<blocks, 256, 0, st>>>(m, first_start, w.key_in, w.idx_in);
    U1GF_CUDA(cudaGetLastError());
    ++launches;
    size_t tb = w.cub_bytes;
    U1GF_CUDA(cub::DeviceRadixSort::SortPairs(w.cub_tmp, tb, w.key_in, w.key_out, w.idx_in, w.perm, (int)m, 0, 64, st));
    merge_gather_kernel<<<blocks, 256, 0, st>>>(m, w.perm, F_rep, sig_rep, w.F_s, w.sig_s, w.status_s, merged_multiplicity);
    U1GF_CUDA(cudaGetLastError());
    ++launches;
    const int rc = u1gf_count_copies(m_, w.F_s, w.sig_s, w.status_s, tol_F, tol_sig, w.id_s, n_merged, w.rep_s, w.mult_s,
                                     nullptr, 0, w.count_ws, w.count_bytes, cuda_stream);
    if (rc != U1GF_OK) return rc;
    launches += t_launches;
    merge_scatter_kernel<<<blocks, 256, 0, st>>>(m, w.perm, w.id_s, w.rep_s, n_merged, first_start, multiplicity, merged_id,
                                                 merged_first_start, merged_multiplicity);
    U1GF_CUDA(cudaGetLastError());
    t_launches = launches + 1;
    return U1GF_OK;
}

}  // extern "C"
