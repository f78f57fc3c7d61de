// orbit.cu -- a1 orbit setup, error plumbing, dispatch of u1gf_relax_batch and the *_host
// convenience entry points of include/u1gf.h.
#include <cmath>
#include <cstring>
#include <new>

#include "u1gf_internal.h"

namespace u1gf {

static thread_local char t_err[512] = "";
thread_local int t_launches = 0;
thread_local cudaEvent_t t_ev0 = nullptr;
thread_local cudaEvent_t t_ev1 = nullptr;
thread_local bool t_ev_valid = false;

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
}

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
    return code;
}

int check_device() {
    static thread_local int cached = 1;  // 1 = unknown
    if (cached != 1) {
        if (cached != U1GF_OK) set_error("no CUDA device of compute capability 10.x (there is no CPU fallback)");
        return cached;
    }
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n < 1) {
        cudaGetLastError();
        cached = U1GF_ENODEV;
        return fail(U1GF_ENODEV, "no CUDA device available (%s); there is no CPU fallback",
                    e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
    }
    int dev = 0;
    cudaGetDevice(&dev);
    int major = 0;
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (major != 10) {
        cached = U1GF_ENODEV;
        return fail(U1GF_ENODEV, "device %d has compute capability %d.x; libu1gf is built for sm_100a only", dev, major);
    }
    cached = U1GF_OK;
    return U1GF_OK;
}

}  // namespace u1gf

using namespace u1gf;

extern "C" {

const char* u1gf_last_error(void) { return t_err; }
int u1gf_abi_version(void) { return 1; }
int32_t u1gf_last_launch_count(void) { return t_launches; }

double u1gf_last_relax_ms(void) {
    if (!t_ev_valid) return -1.0;
    if (cudaEventSynchronize(t_ev1) != cudaSuccess) return -1.0;
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, t_ev0, t_ev1) != cudaSuccess) return -1.0;
    return (double)ms;
}

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

    // one device blob: U | fwd | bwd | order | sgn | lanes-layout links
    auto align = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t bU = align((size_t)V * d * sizeof(double2)), bT = align((size_t)V * d * sizeof(int)),
                 bO = align((size_t)V * sizeof(int)), bS = align((size_t)V);
    const size_t bL = align(lanes_links_bytes(d, D.ext));
    o->blob_bytes = bU + 2 * bT + bO + bS + bL;
    cudaGetDevice(&o->device);
    cudaDeviceGetAttribute(&o->sm_count, cudaDevAttrMultiProcessorCount, o->device);
    cudaError_t e = cudaMalloc(&o->blob, o->blob_bytes);
    if (e != cudaSuccess) {
        delete o;
        return fail(U1GF_ENOMEM, "u1gf_create_orbit: cudaMalloc(%zu): %s", o->blob_bytes, cudaGetErrorString(e));
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
    if (bL) {
        lanes_fill_links(d, D.ext, o->U_host.data(), (double2*)(h + off));
        o->U_lanes = (const double2*)(dptr + off);
        o->U_lanes_host.assign((const double2*)(h + off), (const double2*)(h + off) + (size_t)V * d);
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
    if (!o || which < 0 || which > 2) return fail(U1GF_EINVAL, "u1gf_set_kernel: bad argument");
    o->kernel_choice = which;
    return U1GF_OK;
}

static bool use_lanes(const u1gf_orbit* o) { return o->kernel_choice == 0 && lanes_supported(o); }
static bool use_stream(const u1gf_orbit* o) {
    if (use_lanes(o)) return false;
    return (o->kernel_choice == 0 && stream_preferred(o)) || (o->kernel_choice == 2 && stream_supported(o));
}

const char* u1gf_kernel_name(const u1gf_orbit* o) {
    if (!o) return "";
    return use_lanes(o)    ? lanes_name(o)
           : use_stream(o) ? (o->dev.all_even ? "stream_lane_per_start" : "phased_lane_per_start")
                           : "generic_cta_per_start";
}

size_t u1gf_relax_workspace_bytes(const u1gf_orbit* o, uint64_t n_starts) {
    if (!o) return 0;
    return use_lanes(o)    ? lanes_workspace_bytes(o, n_starts)
           : use_stream(o) ? stream_workspace_bytes(o, n_starts)
                           : generic_workspace_bytes(o, n_starts);
}

int u1gf_relax_batch(const u1gf_orbit* o, uint64_t seed, uint64_t first_start, uint64_t n_starts,
                     const uint64_t* start_ids, double omega, double eps, int32_t max_sweeps, int32_t check_every,
                     double* F_norm, int32_t* sweeps, uint8_t* status, double* sig, double* g_canon, void* workspace,
                     size_t workspace_bytes, void* cuda_stream) {
    t_launches = 0;
    t_ev_valid = false;
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
    if (!t_ev0) {
        U1GF_CUDA(cudaEventCreate(&t_ev0));
        U1GF_CUDA(cudaEventCreate(&t_ev1));
    }
    return use_lanes(o) ? lanes_relax(o, a, st) : use_stream(o) ? stream_relax(o, a, st) : generic_relax(o, a, st);
}

// ---------------------------------------------------------------------------------------------------------
// host-buffer variants: allocate, run, copy back, drain
// ---------------------------------------------------------------------------------------------------------
namespace {
struct DevBuf {
    void* p = nullptr;
    ~DevBuf() {
        if (p) cudaFree(p);
    }
    cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 1); }
};
}  // namespace

int u1gf_relax_batch_host(const u1gf_orbit* o, uint64_t seed, uint64_t first_start, uint64_t n_starts,
                          const uint64_t* start_ids_host, double omega, double eps, int32_t max_sweeps,
                          int32_t check_every, double* F_norm_host, int32_t* sweeps_host, uint8_t* status_host,
                          double* sig_host, double* g_canon_host) {
    if (!o) return fail(U1GF_EINVAL, "u1gf_relax_batch_host: NULL orbit");
    if (int rc = check_device()) return rc;
    if (n_starts == 0) return U1GF_OK;
    const size_t n = (size_t)n_starts, V = (size_t)o->dev.V;
    DevBuf F, sw, stt, sg, gc, ids, ws;
    const size_t wsb = u1gf_relax_workspace_bytes(o, n_starts);
    if (F.alloc(n * 8) || sw.alloc(n * 4) || stt.alloc(n) || sg.alloc(n * 32) || ws.alloc(wsb) ||
        (g_canon_host && gc.alloc(n * V * 16)) || (start_ids_host && ids.alloc(n * 8))) {
        cudaGetLastError();
        return fail(U1GF_ENOMEM, "u1gf_relax_batch_host: device allocation failed");
    }
    if (start_ids_host) U1GF_CUDA(cudaMemcpy(ids.p, start_ids_host, n * 8, cudaMemcpyHostToDevice));
    int rc = u1gf_relax_batch(o, seed, first_start, n_starts, start_ids_host ? (const uint64_t*)ids.p : nullptr, omega,
                              eps, max_sweeps, check_every, (double*)F.p, (int32_t*)sw.p, (uint8_t*)stt.p,
                              (double*)sg.p, g_canon_host ? (double*)gc.p : nullptr, ws.p, wsb, nullptr);
    if (rc) return rc;
    if (F_norm_host) U1GF_CUDA(cudaMemcpy(F_norm_host, F.p, n * 8, cudaMemcpyDeviceToHost));
    if (sweeps_host) U1GF_CUDA(cudaMemcpy(sweeps_host, sw.p, n * 4, cudaMemcpyDeviceToHost));
    if (status_host) U1GF_CUDA(cudaMemcpy(status_host, stt.p, n, cudaMemcpyDeviceToHost));
    if (sig_host) U1GF_CUDA(cudaMemcpy(sig_host, sg.p, n * 32, cudaMemcpyDeviceToHost));
    if (g_canon_host) U1GF_CUDA(cudaMemcpy(g_canon_host, gc.p, n * V * 16, cudaMemcpyDeviceToHost));
    U1GF_CUDA(cudaDeviceSynchronize());
    return U1GF_OK;
}

int u1gf_check_fp_host(const u1gf_orbit* o, uint64_t n_cfg, const double* g_host, double tol_fp,
                       double* lambda1_host, uint8_t* region_host, int64_t* n_in_region_host) {
    if (!o || !g_host) return fail(U1GF_EINVAL, "u1gf_check_fp_host: NULL argument");
    if (int rc = check_device()) return rc;
    const size_t n = (size_t)n_cfg, V = (size_t)o->dev.V;
    DevBuf g, lam, reg, cnt;
    if (g.alloc(n * V * 16) || lam.alloc(n * 8) || reg.alloc(n) || cnt.alloc(8)) {
        cudaGetLastError();
        return fail(U1GF_ENOMEM, "u1gf_check_fp_host: device allocation failed");
    }
    U1GF_CUDA(cudaMemcpy(g.p, g_host, n * V * 16, cudaMemcpyHostToDevice));
    int rc = u1gf_check_fp(o, n_cfg, (const double*)g.p, tol_fp, (double*)lam.p, (uint8_t*)reg.p, (int64_t*)cnt.p,
                           nullptr);
    if (rc) return rc;
    if (lambda1_host) U1GF_CUDA(cudaMemcpy(lambda1_host, lam.p, n * 8, cudaMemcpyDeviceToHost));
    if (region_host) U1GF_CUDA(cudaMemcpy(region_host, reg.p, n, cudaMemcpyDeviceToHost));
    if (n_in_region_host) U1GF_CUDA(cudaMemcpy(n_in_region_host, cnt.p, 8, cudaMemcpyDeviceToHost));
    U1GF_CUDA(cudaDeviceSynchronize());
    return U1GF_OK;
}

int u1gf_count_copies_host(uint64_t n_, const double* F_norm_host, const double* sig_host, const uint8_t* status_host,
                           double tol_F, double tol_sig, int32_t* copy_id_host, int64_t* n_distinct_host,
                           int64_t* rep_host, int64_t* multiplicity_host, int64_t* hist_host, int32_t nbins) {
    if (n_ && (!F_norm_host || !sig_host || !status_host))
        return fail(U1GF_EINVAL, "u1gf_count_copies_host: NULL input array");
    if (int rc = check_device()) return rc;
    const size_t n = (size_t)n_;
    DevBuf F, sg, stt, cid, nd, rep, mul, hist, ws;
    const size_t wsb = u1gf_count_workspace_bytes(n_);
    if (F.alloc(n * 8) || sg.alloc(n * 32) || stt.alloc(n) || cid.alloc(n * 4) || nd.alloc(8) || rep.alloc(n * 8) ||
        mul.alloc(n * 8) || hist.alloc((size_t)(nbins > 0 ? nbins : 0) * 8) || ws.alloc(wsb)) {
        cudaGetLastError();
        return fail(U1GF_ENOMEM, "u1gf_count_copies_host: device allocation failed");
    }
    if (n) {
        U1GF_CUDA(cudaMemcpy(F.p, F_norm_host, n * 8, cudaMemcpyHostToDevice));
        U1GF_CUDA(cudaMemcpy(sg.p, sig_host, n * 32, cudaMemcpyHostToDevice));
        U1GF_CUDA(cudaMemcpy(stt.p, status_host, n, cudaMemcpyHostToDevice));
    }
    int rc = u1gf_count_copies(n_, (const double*)F.p, (const double*)sg.p, (const uint8_t*)stt.p, tol_F, tol_sig,
                               (int32_t*)cid.p, (int64_t*)nd.p, (int64_t*)rep.p, (int64_t*)mul.p,
                               nbins > 0 ? (int64_t*)hist.p : nullptr, nbins, ws.p, wsb, nullptr);
    if (rc) return rc;
    int64_t ndh = 0;
    U1GF_CUDA(cudaMemcpy(&ndh, nd.p, 8, cudaMemcpyDeviceToHost));
    if (n_distinct_host) *n_distinct_host = ndh;
    if (copy_id_host && n) U1GF_CUDA(cudaMemcpy(copy_id_host, cid.p, n * 4, cudaMemcpyDeviceToHost));
    if (rep_host && ndh) U1GF_CUDA(cudaMemcpy(rep_host, rep.p, (size_t)ndh * 8, cudaMemcpyDeviceToHost));
    if (multiplicity_host && ndh)
        U1GF_CUDA(cudaMemcpy(multiplicity_host, mul.p, (size_t)ndh * 8, cudaMemcpyDeviceToHost));
    if (hist_host && nbins > 0) U1GF_CUDA(cudaMemcpy(hist_host, hist.p, (size_t)nbins * 8, cudaMemcpyDeviceToHost));
    U1GF_CUDA(cudaDeviceSynchronize());
    return U1GF_OK;
}

}  // extern "C"
