// orbit.cu -- a1 orbit setup, dispatch of u1gf_relax_batch and the *_host convenience entry points
// of include/u1gf.h (error plumbing: common.cu).
#include <cmath>
#include <cstring>
#include <new>

#include "u1gf_internal.h"

using namespace u1gf;

extern "C" {

int32_t u1gf_orbit_volume(const u1gf_orbit* o) { return o ? o->dev.V : 0; }
int32_t u1gf_orbit_dim(const u1gf_orbit* o) { return o ? o->dev.d : 0; }

int u1gf_create_orbit(int d, const int32_t* extents, const double* theta_host, u1gf_orbit** out) {
    t_launches = 0;
    if (out) *out = nullptr;
    if (!out || !extents || !theta_host) return fail(U1GF_EINVAL, "u1gf_create_orbit: NULL argument");
    if (d < 1 || d > 4) return fail(U1GF_EINVAL, "u1gf_create_orbit: d = %d outside 1..4", d);
    long V = 1;
    for (int mu = 0; mu < d; ++mu) {
        if (extents[mu] < 2) return fail(U1GF_EINVAL, "u1gf_create_orbit: extent[%d] = %d < 2", mu, extents[mu]);
        V *= extents[mu];
        if (V > kMaxV) return fail(U1GF_EINVAL, "u1gf_create_orbit: volume exceeds %d sites", kMaxV);
    }
    for (long l = 0; l < V * d; ++l)
        if (!std::isfinite(theta_host[l])) return fail(U1GF_EINVAL, "u1gf_create_orbit: theta[%ld] is not finite", l);
    if (int rc = check_device()) return rc;

    u1gf_orbit* o = new (std::nothrow) u1gf_orbit();
    if (!o) return fail(U1GF_ENOMEM, "u1gf_create_orbit: host allocation failed");
    OrbitDev& D = o->dev;
    D.d = d;
    D.V = (int)V;
    int n_odd = 0;
    for (int mu = 0; mu < 4; ++mu) {
        D.ext[mu] = mu < d ? extents[mu] : 1;
        if (mu < d && (extents[mu] & 1)) ++n_odd;
    }
    D.all_even = n_odd == 0;

    // geometry tables
    std::vector<int> fwd(V * d), bwd(V * d), phase(V), order(V);
    std::vector<uint8_t> sgn(V);
    for (int i = 0; i < V; ++i) {
        int x[4], r = i, par = 0, lvl = 0, stride = 1;
        for (int mu = 0; mu < d; ++mu) {
            x[mu] = r % D.ext[mu];
            r /= D.ext[mu];
            par += x[mu];
            if ((D.ext[mu] & 1) && x[mu] == D.ext[mu] - 1) ++lvl;  // level of R3
        }
        for (int mu = 0; mu < d; ++mu) {
            const int n = D.ext[mu];
            fwd[i * d + mu] = i + (((x[mu] + 1) % n) - x[mu]) * stride;
            bwd[i * d + mu] = i + (((x[mu] + n - 1) % n) - x[mu]) * stride;
            stride *= n;
        }
        phase[i] = (par & 1) * (n_odd + 1) + lvl;
        uint8_t bits = 0;
        for (int k = 0; k < 4; ++k) {  // signature signs: Philox key (0x51,0), counter (i,k,0,1)
            const u32x4 w = philox((uint32_t)i, (uint32_t)k, 0u, 1u, 0x51u, 0u);
            if (w.x & 1u) bits |= (uint8_t)(1u << k);
            if (w.y & 1u) bits |= (uint8_t)(1u << (4 + k));
        }
        sgn[i] = bits;
    }
    std::vector<uint8_t> fin(V);
    for (int i = 0; i < V; ++i) {
        bool last = true;
        for (int mu = 0; mu < d; ++mu) last = last && phase[fwd[i * d + mu]] < phase[i] && phase[bwd[i * d + mu]] < phase[i];
        fin[i] = last ? 1 : 0;
    }
    // phases in order, empty ones dropped
    D.n_phases = 0;
    D.phase_off[0] = 0;
    D.max_phase = 0;
    int pos = 0;
    for (int p = 0; p < 2 * (n_odd + 1); ++p) {
        const int begin = pos;
        for (int i = 0; i < V; ++i)
            if (phase[i] == p) order[pos++] = i;
        if (pos > begin) {
            D.phase_off[++D.n_phases] = pos;
            if (pos - begin > D.max_phase) D.max_phase = pos - begin;
        }
    }

    // links on the host with libm, interleaved (cos, sin)
    o->U_host.resize((size_t)V * d * 2);
    for (long l = 0; l < V * d; ++l) {
        o->U_host[2 * l] = std::cos(theta_host[l]);
        o->U_host[2 * l + 1] = std::sin(theta_host[l]);
    }

    // one device blob: U | fwd | bwd | order | sgn | fin | lanes-layout links | TMA-layout links
    auto align = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t bU = align((size_t)V * d * sizeof(double2)), bT = align((size_t)V * d * sizeof(int)),
                 bO = align((size_t)V * sizeof(int)), bS = align((size_t)V);
    const size_t bL = align(lanes_links_bytes(d, D.ext)), bM = align(tma_links_bytes(d, D.ext));
    o->blob_bytes = bU + 2 * bT + bO + 2 * bS + bL + bM;
    cudaGetDevice(&o->device);
    cudaDeviceGetAttribute(&o->sm_count, cudaDevAttrMultiProcessorCount, o->device);
    cudaError_t e = cudaMalloc(&o->blob, o->blob_bytes);
    if (e != cudaSuccess) {
        const size_t bytes = o->blob_bytes;
        delete o;
        return fail(U1GF_ENOMEM, "u1gf_create_orbit: cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e));
    }
    std::vector<char> host(o->blob_bytes, 0);
    char* h = host.data();
    char* dptr = (char*)o->blob;
    size_t off = 0;
    std::memcpy(h + off, o->U_host.data(), (size_t)V * d * sizeof(double2));
    D.U = (const double2*)(dptr + off);
    off += bU;
    std::memcpy(h + off, fwd.data(), (size_t)V * d * sizeof(int));
    D.fwd = (const int*)(dptr + off);
    off += bT;
    std::memcpy(h + off, bwd.data(), (size_t)V * d * sizeof(int));
    D.bwd = (const int*)(dptr + off);
    off += bT;
    std::memcpy(h + off, order.data(), (size_t)V * sizeof(int));
    D.order = (const int*)(dptr + off);
    off += bO;
    std::memcpy(h + off, sgn.data(), (size_t)V);
    D.sgn = (const uint8_t*)(dptr + off);
    off += bS;
    std::memcpy(h + off, fin.data(), (size_t)V);
    D.fin = (const uint8_t*)(dptr + off);
    off += bS;
    if (bL) {
        lanes_fill_links(d, D.ext, o->U_host.data(), (double2*)(h + off));
        o->U_lanes = (const double2*)(dptr + off);
        o->U_lanes_host.assign((const double2*)(h + off), (const double2*)(h + off) + (size_t)V * d);
    }
    off += bL;
    if (bM) {
        tma_fill_links(o, (double2*)(h + off));
        o->U_tma = (const double2*)(dptr + off);
    }
    e = cudaMemcpy(o->blob, h, o->blob_bytes, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(o->blob);
        delete o;
        return fail(U1GF_ECUDA, "u1gf_create_orbit: cudaMemcpy: %s", cudaGetErrorString(e));
    }
    *out = o;
    return U1GF_OK;
}

int u1gf_destroy_orbit(u1gf_orbit* o) {
    if (!o) return U1GF_OK;
    cudaError_t e = cudaFree(o->blob);
    delete o;
    if (e != cudaSuccess) return fail(U1GF_ECUDA, "u1gf_destroy_orbit: cudaFree: %s", cudaGetErrorString(e));
    return U1GF_OK;
}

int u1gf_set_kernel(u1gf_orbit* o, int32_t which) {
    if (!o || which < 0 || which > 3) return fail(U1GF_EINVAL, "u1gf_set_kernel: bad argument");
    o->kernel_choice = which;
    return U1GF_OK;
}

static bool use_lanes(const u1gf_orbit* o) { return o->kernel_choice == 0 && lanes_supported(o); }
static bool use_tma(const u1gf_orbit* o) {
    return !use_lanes(o) && (o->kernel_choice == 0 || o->kernel_choice == 3) && tma_supported(o);
}
static bool use_stream(const u1gf_orbit* o) {
    if (use_lanes(o) || use_tma(o)) return false;
    return (o->kernel_choice == 0 && stream_preferred(o)) || (o->kernel_choice == 2 && stream_supported(o));
}

const char* u1gf_kernel_name(const u1gf_orbit* o) {
    if (!o) return "";
    return use_lanes(o)    ? lanes_name(o)
           : use_tma(o)    ? "tma_stream_lane_per_start"
           : use_stream(o) ? (o->dev.all_even ? "stream_lane_per_start" : "phased_lane_per_start")
                           : "generic_cta_per_start";
}

size_t u1gf_relax_workspace_bytes(const u1gf_orbit* o, uint64_t n_starts) {
    if (!o) return 0;
    return use_lanes(o)    ? lanes_workspace_bytes(o, n_starts)
           : use_tma(o)    ? tma_workspace_bytes(o, n_starts)
           : use_stream(o) ? stream_workspace_bytes(o, n_starts)
                           : generic_workspace_bytes(o, n_starts);
}

int u1gf_relax_batch(const u1gf_orbit* o, uint64_t seed, uint64_t first_start, uint64_t n_starts,
                     const uint64_t* start_ids, double omega, double eps, int32_t max_sweeps, int32_t check_every,
                     double* F_norm, int32_t* sweeps, uint8_t* status, double* sig, double* g_canon, void* workspace,
                     size_t workspace_bytes, void* cuda_stream) {
    t_launches = 0;
    if (!o) return fail(U1GF_EINVAL, "u1gf_relax_batch: NULL orbit");
    if (!(omega >= 1.0 && omega < 2.0)) return fail(U1GF_EINVAL, "u1gf_relax_batch: omega = %g outside [1,2)", omega);
    if (!(eps > 0.0)) return fail(U1GF_EINVAL, "u1gf_relax_batch: eps = %g must be > 0", eps);
    if (max_sweeps < 1 || check_every < 1)
        return fail(U1GF_EINVAL, "u1gf_relax_batch: max_sweeps and check_every must be >= 1");
    if (n_starts == 0) return U1GF_OK;
    if (n_starts > (1ull << 40)) return fail(U1GF_EINVAL, "u1gf_relax_batch: n_starts too large");
    if (!F_norm || !sweeps || !status || !sig) return fail(U1GF_EINVAL, "u1gf_relax_batch: NULL output array");
    if (int rc = check_device()) return rc;
    const size_t need = u1gf_relax_workspace_bytes(o, n_starts);
    if (!workspace || workspace_bytes < need)
        return fail(U1GF_ENOMEM, "u1gf_relax_batch: workspace of %zu bytes needed, %zu given", need, workspace_bytes);
    if (((uintptr_t)workspace & 255) != 0) return fail(U1GF_EINVAL, "u1gf_relax_batch: workspace not 256-byte aligned");
    RelaxArgs a{seed, first_start, n_starts, start_ids, omega, eps, max_sweeps, check_every,
                F_norm, sweeps, status, sig, g_canon, workspace, workspace_bytes};
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return use_lanes(o)    ? lanes_relax(o, a, st)
           : use_tma(o)    ? tma_relax(o, a, st)
           : use_stream(o) ? stream_relax(o, a, st)
                           : generic_relax(o, a, st);
}

}  // extern "C"
