// ensemble.cu -- SURVEY section 8(f)-3: many gauge orbits of one lattice shape relaxed in ONE kernel launch.
// The paper's workload is an ensemble: 100 orbits x 4 mebisamples per lattice size (Tab. I, Tab. III
// L213-220), one lattice per thread block with the grid over samples (L121).  Here the resident lane-per-start kernels
// (relax_lanes.cu) number their 32-start batches over all orbits of the ensemble; a team of 32 lanes works through its
// batches orbit by orbit and reloads the link table in shared memory at an orbit boundary.  De-duplication is per
// orbit (copies of different orbits are unrelated): in one pass with the orbit index as the major sort key when the caller's
// workspace is large enough for all records (count_copies.cu), else as a loop over u1gf_count_copies on the orbits' slices.
// Shapes without a resident kernel (2x2, 6x6, 2^3, 8^3, odd extents, ...) run on the generic kernel, one CTA per start
// with the grid over the starts of all orbits -- the paper's own mapping.
#include <new>

#include "u1gf_internal.h"

struct u1gf_ensemble {
    std::vector<u1gf_orbit*> orbits;            // members (library-owned); all of one shape
    void* blob = nullptr;                       // [n_orbits][lanes_stride] double2 tables, then the seeds
    const double2* U_all = nullptr;
    const unsigned long long* seeds_dev = nullptr;
    unsigned long long lanes_stride = 0;        // double2 elements per orbit
    bool generic = false;                       // no resident kernel for the shape: plain link tables [V*d] per orbit and
                                                // the generic kernel, one CTA per start (the paper's mapping, L121)
};

using namespace u1gf;

extern "C" {

int u1gf_destroy_ensemble(u1gf_ensemble* e) {
    if (!e) return U1GF_OK;
    for (u1gf_orbit* o : e->orbits) u1gf_destroy_orbit(o);
    cudaError_t err = e->blob ? cudaFree(e->blob) : cudaSuccess;
    delete e;
    if (err != cudaSuccess) return fail(U1GF_ECUDA, "u1gf_destroy_ensemble: cudaFree: %s", cudaGetErrorString(err));
    return U1GF_OK;
}

int u1gf_create_ensemble(int d, const int32_t* extents, int32_t n_orbits, const double* theta_host,
                         const uint64_t* seeds_host, u1gf_ensemble** out) {
    t_launches = 0;
    if (out) *out = nullptr;
    if (!out || !extents || !theta_host || !seeds_host) return fail(U1GF_EINVAL, "u1gf_create_ensemble: NULL argument");
    if (n_orbits < 1 || n_orbits > (1 << 20)) return fail(U1GF_EINVAL, "u1gf_create_ensemble: n_orbits = %d outside 1..2^20", n_orbits);
    u1gf_ensemble* e = new (std::nothrow) u1gf_ensemble;
    if (!e) return fail(U1GF_ENOMEM, "u1gf_create_ensemble: out of host memory");
    size_t Vd = 0;
    for (int k = 0; k < n_orbits; ++k) {
        u1gf_orbit* o = nullptr;
        const int rc = u1gf_create_orbit(d, extents, theta_host + (size_t)k * Vd, &o);
        if (rc != U1GF_OK) {
            u1gf_destroy_ensemble(e);
            return rc;   // message set by u1gf_create_orbit
        }
        e->orbits.push_back(o);
        Vd = (size_t)o->dev.V * (size_t)o->dev.d;
    }
    const u1gf_orbit* o0 = e->orbits[0];
    e->generic = !lanes_supported(o0);
    const size_t tab_bytes = e->generic ? Vd * sizeof(double2) : lanes_links_bytes(o0->dev.d, o0->dev.ext);
    e->lanes_stride = tab_bytes / sizeof(double2);
    const size_t seeds_off = ((size_t)n_orbits * tab_bytes + 255) & ~(size_t)255;
    cudaError_t err = cudaMalloc(&e->blob, seeds_off + (size_t)n_orbits * sizeof(uint64_t));
    if (err != cudaSuccess) {
        u1gf_destroy_ensemble(e);
        return fail(U1GF_ENOMEM, "u1gf_create_ensemble: cudaMalloc: %s", cudaGetErrorString(err));
    }
    e->U_all = (const double2*)e->blob;
    e->seeds_dev = (const unsigned long long*)((char*)e->blob + seeds_off);
    for (int k = 0; k < n_orbits && err == cudaSuccess; ++k)   // the members' tables, device to device
        err = cudaMemcpy((char*)e->blob + (size_t)k * tab_bytes,
                         e->generic ? (const void*)e->orbits[k]->dev.U : (const void*)e->orbits[k]->U_lanes, tab_bytes,
                         cudaMemcpyDeviceToDevice);
    if (err == cudaSuccess)
        err = cudaMemcpy((char*)e->blob + seeds_off, seeds_host, (size_t)n_orbits * sizeof(uint64_t), cudaMemcpyHostToDevice);
    if (err != cudaSuccess) {
        u1gf_destroy_ensemble(e);
        return fail(U1GF_ECUDA, "u1gf_create_ensemble: cudaMemcpy: %s", cudaGetErrorString(err));
    }
    *out = e;
    return U1GF_OK;
}

int32_t u1gf_ensemble_size(const u1gf_ensemble* e) { return e ? (int32_t)e->orbits.size() : 0; }

const u1gf_orbit* u1gf_ensemble_orbit(const u1gf_ensemble* e, int32_t k) {
    if (!e || k < 0 || (size_t)k >= e->orbits.size()) return nullptr;
    return e->orbits[(size_t)k];
}

size_t u1gf_relax_ensemble_workspace_bytes(const u1gf_ensemble* e, uint64_t n_starts_per_orbit) {
    if (!e) return 0;
    if (e->generic) return generic_workspace_bytes(e->orbits[0], n_starts_per_orbit);
    return lanes_ens_workspace_bytes(e->orbits[0], (unsigned)e->orbits.size(), n_starts_per_orbit);
}

int u1gf_relax_ensemble(const u1gf_ensemble* e, uint64_t first_start, uint64_t n_starts_per_orbit, double omega,
                        double eps, int32_t max_sweeps, int32_t check_every, double* F_norm, int32_t* sweeps,
                        uint8_t* status, double* sig, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    t_launches = 0;
    if (!e) return fail(U1GF_EINVAL, "u1gf_relax_ensemble: NULL ensemble");
    if (!(omega >= 1.0 && omega < 2.0)) return fail(U1GF_EINVAL, "u1gf_relax_ensemble: omega = %g outside [1,2)", omega);
    if (!(eps > 0.0)) return fail(U1GF_EINVAL, "u1gf_relax_ensemble: eps = %g must be > 0", eps);
    if (max_sweeps < 1 || check_every < 1)
        return fail(U1GF_EINVAL, "u1gf_relax_ensemble: max_sweeps and check_every must be >= 1");
    if (n_starts_per_orbit == 0) return U1GF_OK;
    if (n_starts_per_orbit > (1ull << 40) / e->orbits.size()) return fail(U1GF_EINVAL, "u1gf_relax_ensemble: too many starts");
    if (!F_norm || !sweeps || !status || !sig) return fail(U1GF_EINVAL, "u1gf_relax_ensemble: NULL output array");
    if (int rc = check_device()) return rc;
    const size_t need = u1gf_relax_ensemble_workspace_bytes(e, n_starts_per_orbit);
    if (!workspace || workspace_bytes < need)
        return fail(U1GF_ENOMEM, "u1gf_relax_ensemble: workspace of %zu bytes needed, %zu given", need, workspace_bytes);
    if (((uintptr_t)workspace & 255) != 0) return fail(U1GF_EINVAL, "u1gf_relax_ensemble: workspace not 256-byte aligned");
    RelaxArgs a{0, first_start, n_starts_per_orbit, nullptr, omega, eps, max_sweeps, check_every,
                F_norm, sweeps, status, sig, nullptr, workspace, workspace_bytes};
    if (e->generic)
        return generic_relax_ens(e->orbits[0], e->U_all, e->seeds_dev, (unsigned)e->orbits.size(), a, (cudaStream_t)cuda_stream);
    return lanes_relax_ens(e->orbits[0], e->U_all, e->lanes_stride, e->seeds_dev, (unsigned)e->orbits.size(), a,
                           (cudaStream_t)cuda_stream);
}

size_t u1gf_count_ensemble_workspace_bytes(uint64_t n_per_orbit) { return u1gf_count_workspace_bytes(n_per_orbit); }
size_t u1gf_count_ensemble_onepass_workspace_bytes(int32_t n_orbits, uint64_t n_per_orbit) {
    return n_orbits > 1 ? count_ens_onepass_workspace_bytes((unsigned)n_orbits, n_per_orbit) : 0;
}

int u1gf_count_copies_ensemble(int32_t n_orbits, uint64_t n_per_orbit, const double* F_norm, const double* sig,
                               const uint8_t* status, double tol_F, double tol_sig, int32_t* copy_id,
                               int64_t* n_distinct, int64_t* rep, int64_t* multiplicity, int64_t* hist, int32_t nbins,
                               void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (n_orbits < 0) return fail(U1GF_EINVAL, "u1gf_count_copies_ensemble: n_orbits < 0");
    // one pass over all orbits when the workspace is large enough for it (u1gf_count_ensemble_onepass_workspace_bytes)
    const size_t onepass = n_orbits > 1 ? count_ens_onepass_workspace_bytes((unsigned)n_orbits, n_per_orbit) : 0;
    if (onepass && workspace && workspace_bytes >= onepass) {
        t_launches = 0;
        if (!n_distinct || !F_norm || !sig || !status || !copy_id || !rep || !multiplicity)
            return fail(U1GF_EINVAL, "u1gf_count_copies_ensemble: NULL array");
        if (hist && nbins < 1) return fail(U1GF_EINVAL, "u1gf_count_copies_ensemble: nbins must be >= 1 when hist is given");
        if (hist && (unsigned long long)n_orbits * (unsigned long long)nbins >= (1ull << 31))
            return fail(U1GF_EINVAL, "u1gf_count_copies_ensemble: n_orbits * nbins must be below 2^31");
        if (!(tol_F >= 0.0) || !(tol_sig >= 0.0)) return fail(U1GF_EINVAL, "u1gf_count_copies_ensemble: negative tolerance");
        if (((uintptr_t)workspace & 255) != 0) return fail(U1GF_EINVAL, "u1gf_count_copies_ensemble: workspace not 256-byte aligned");
        if (int rc = check_device()) return rc;
        return count_copies_ens_onepass((unsigned)n_orbits, (unsigned)n_per_orbit, F_norm, sig, status, tol_F, tol_sig, copy_id,
                                        n_distinct, rep, multiplicity, hist, nbins, workspace, (cudaStream_t)cuda_stream);
    }
    int launches = 0;
    const size_t n = (size_t)n_per_orbit;
    for (int32_t k = 0; k < n_orbits; ++k) {   // the same workspace serves the orbits one after the other (stream order)
        const size_t off = (size_t)k * n;
        const int rc = u1gf_count_copies(n_per_orbit, F_norm ? F_norm + off : nullptr, sig ? sig + 4 * off : nullptr,
                                         status ? status + off : nullptr, tol_F, tol_sig, copy_id ? copy_id + off : nullptr,
                                         n_distinct ? n_distinct + k : nullptr, rep ? rep + off : nullptr,
                                         multiplicity ? multiplicity + off : nullptr,
                                         hist ? hist + (size_t)k * (size_t)(nbins > 0 ? nbins : 0) : nullptr, nbins,
                                         workspace, workspace_bytes, cuda_stream);
        if (rc != U1GF_OK) return rc;
        launches += t_launches;
    }
    t_launches = launches;
    return U1GF_OK;
}

}  // extern "C"
