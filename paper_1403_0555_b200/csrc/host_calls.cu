// host_calls.cu -- the *_host entry points of include/u1gf.h: host result buffers, device scratch from a per-thread
// arena, copies inside the call, stream drained before returning.  u1gf_pipeline_host is the whole hot path in one call
// (what bench.py's e2e leg times): relax -> count -> fields of the representatives (relaxed once more on cold orbits, kept
// from the first pass on hot ones) -> first-Gribov-region test, with every intermediate staying on the device.
#include <algorithm>
#include <vector>

#include "u1gf_internal.h"

using namespace u1gf;

namespace {

// Device scratch of the *_host entry points: one grow-only allocation per host thread, carved up by every call and
// kept between calls (u1gf_release_host_scratch frees it), so that a call's timed path holds copies and kernels, not
// cudaMalloc / cudaFree.
struct Arena {
    char* base = nullptr;
    size_t cap = 0, used = 0;
    int device = -1;   // the device `base` was allocated on: a thread that switches device gets a fresh allocation there
    ~Arena() {
        // at thread exit; at process exit the runtime may already be gone, then cudaFree reports an error we drop
        if (base) cudaFree(base);
    }
    void release() {
        if (base) cudaFree(base);   // a device pointer identifies its own device: no cudaSetDevice needed
        base = nullptr;
        cap = used = 0;
        device = -1;
    }
    bool reserve(size_t bytes) {
        used = 0;
        int dev = -1;
        if (cudaGetDevice(&dev) != cudaSuccess) {
            cudaGetLastError();
            return false;
        }
        if (base && dev == device && bytes <= cap) return true;
        release();
        if (cudaMalloc((void**)&base, bytes) != cudaSuccess) {
            cudaGetLastError();
            base = nullptr;
            return false;
        }
        cap = bytes;
        device = dev;
        return true;
    }
    void* take(size_t bytes) {
        void* p = base + used;
        used += (bytes + 255) & ~(size_t)255;
        return p;
    }
    static size_t padded(size_t bytes) { return (bytes + 255) & ~(size_t)255; }
};
thread_local Arena t_arena;

// The tables of an orbit live on the device that was current in u1gf_create_orbit; the *_host calls allocate and launch
// on the current device, so the two must agree.
int same_device(const u1gf_orbit* o, const char* who) {
    int dev = -1;
    U1GF_CUDA(cudaGetDevice(&dev));
    if (dev != o->device)
        return fail(U1GF_EINVAL, "%s: the orbit was created on device %d, the current device is %d", who, o->device, dev);
    return U1GF_OK;
}

// Error returns of u1gf_pipeline_host must not leave copies into the caller's host arrays in flight.
struct DrainUnlessDone {
    bool done = false;
    ~DrainUnlessDone() {
        if (!done) cudaDeviceSynchronize();
    }
};

struct DevBuf {   // a slice of the arena
    void* p = nullptr;
    void take(size_t bytes) { p = t_arena.take(bytes ? bytes : 1); }
};

__global__ void add_offset_kernel(unsigned long long n, const int64_t* __restrict__ in, unsigned long long off, uint64_t* out) {
    for (unsigned long long k = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; k < n;
         k += (unsigned long long)gridDim.x * blockDim.x)
        out[k] = (uint64_t)in[k] + off;
}

__global__ void gather_F_kernel(unsigned long long n, const int64_t* __restrict__ rep, const double* __restrict__ F, double* out) {
    for (unsigned long long k = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; k < n;
         k += (unsigned long long)gridDim.x * blockDim.x)
        out[k] = F[rep[k]];
}

}  // namespace

extern "C" {

int u1gf_release_host_scratch(void) {
    t_arena.release();
    return U1GF_OK;
}

int u1gf_relax_batch_host(const u1gf_orbit* o, uint64_t seed, uint64_t first_start, uint64_t n_starts,
                          const uint64_t* start_ids_host, double omega, double eps, int32_t max_sweeps,
                          int32_t check_every, double* F_norm_host, int32_t* sweeps_host, uint8_t* status_host,
                          double* sig_host, double* g_canon_host) {
    if (!o) return fail(U1GF_EINVAL, "u1gf_relax_batch_host: NULL orbit");
    if (int rc = check_device()) return rc;
    if (int rc = same_device(o, "u1gf_relax_batch_host")) return rc;
    if (n_starts == 0) return U1GF_OK;
    const size_t n = (size_t)n_starts, V = (size_t)o->dev.V;
    DevBuf F, sw, stt, sg, gc, ids, ws;
    const size_t wsb = u1gf_relax_workspace_bytes(o, n_starts);
    if (!t_arena.reserve(Arena::padded(n * 8) + Arena::padded(n * 4) + Arena::padded(n) + Arena::padded(n * 32) +
                         Arena::padded(wsb) + (g_canon_host ? Arena::padded(n * V * 16) : 0) +
                         (start_ids_host ? Arena::padded(n * 8) : 0) + 1024))
        return fail(U1GF_ENOMEM, "u1gf_relax_batch_host: device allocation failed");
    F.take(n * 8); sw.take(n * 4); stt.take(n); sg.take(n * 32); ws.take(wsb);
    if (g_canon_host) gc.take(n * V * 16);
    if (start_ids_host) ids.take(n * 8);
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
    if (int rc = same_device(o, "u1gf_check_fp_host")) return rc;
    const size_t n = (size_t)n_cfg, V = (size_t)o->dev.V;
    DevBuf g, lam, reg, cnt;
    if (!t_arena.reserve(Arena::padded(n * V * 16) + Arena::padded(n * 8) + Arena::padded(n) + 1024))
        return fail(U1GF_ENOMEM, "u1gf_check_fp_host: device allocation failed");
    g.take(n * V * 16); lam.take(n * 8); reg.take(n); cnt.take(8);
    U1GF_CUDA(cudaMemcpy(g.p, g_host, n * V * 16, cudaMemcpyHostToDevice));
    int rc = u1gf_check_fp(o, n_cfg, (const double*)g.p, nullptr, tol_fp, (double*)lam.p, (uint8_t*)reg.p,
                           (int64_t*)cnt.p, nullptr, nullptr);
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
    const size_t hb = (size_t)(nbins > 0 ? nbins : 0) * 8;
    if (!t_arena.reserve(2 * Arena::padded(n * 8) + Arena::padded(n * 32) + Arena::padded(n) + Arena::padded(n * 4) +
                         Arena::padded(n * 8) + Arena::padded(hb) + Arena::padded(wsb) + 2048))
        return fail(U1GF_ENOMEM, "u1gf_count_copies_host: device allocation failed");
    F.take(n * 8); sg.take(n * 32); stt.take(n); cid.take(n * 4); nd.take(8); rep.take(n * 8); mul.take(n * 8);
    hist.take(hb); ws.take(wsb);
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


int u1gf_pipeline_host(const u1gf_orbit* o, uint64_t seed, uint64_t first_start, uint64_t n_starts, double omega,
                       double eps, int32_t max_sweeps, int32_t check_every, double tol_F, double tol_sig, double tol_fp,
                       int32_t nbins, double* F_norm_host, int32_t* sweeps_host, uint8_t* status_host, double* sig_host,
                       int32_t* copy_id_host, int64_t copy_capacity, int64_t* n_distinct_host, int64_t* rep_host,
                       int64_t* multiplicity_host, double* F_rep_host, double* lambda1_host, uint8_t* region_host,
                       int64_t* n_in_region_host, int64_t* hist_host) {
    if (!o) return fail(U1GF_EINVAL, "u1gf_pipeline_host: NULL orbit");
    if (!n_distinct_host || !n_in_region_host) return fail(U1GF_EINVAL, "u1gf_pipeline_host: NULL count output");
    if (copy_capacity < 0 || nbins < 0) return fail(U1GF_EINVAL, "u1gf_pipeline_host: negative capacity");
    if (n_starts >= (1ull << 31)) return fail(U1GF_EINVAL, "u1gf_pipeline_host: n_starts must be below 2^31");
    if (int rc = check_device()) return rc;
    if (int rc = same_device(o, "u1gf_pipeline_host")) return rc;
    *n_distinct_host = 0;
    *n_in_region_host = 0;
    if (n_starts == 0) return U1GF_OK;
    const size_t n = (size_t)n_starts, V = (size_t)o->dev.V;
    // Where do the fields of the representatives come from?  Cold orbits (few copies): the representatives are relaxed once
    // more, with their fields written out, in chunks whose fields fit a fixed budget.  Hot orbits (most starts are their own
    // copy; the previous call on this handle found n_distinct > n/4): the first pass writes the fields of ALL starts and
    // u1gf_check_fp picks the representatives through cfg_index = rep -- nothing is relaxed twice.  The results are the same
    // either way: a start is a pure function of its index.
    const size_t g_budget = (size_t)1 << 30;
    size_t chunk = std::max<size_t>(1, g_budget / (V * 16));
    if (chunk > n) chunk = n;
    const size_t n_chunks = (n + chunk - 1) / chunk;
    bool keep = false;
    if (o->pipeline_keep_fields) {
        size_t free_b = 0, total_b = 0;
        U1GF_CUDA(cudaMemGetInfo(&free_b, &total_b));
        keep = n * V * 16 <= total_b / 4;
    }
    const size_t ws_relax = u1gf_relax_workspace_bytes(o, n_starts), ws_count = u1gf_count_workspace_bytes(n_starts);
    const size_t ws = std::max(ws_relax, ws_count);
    const size_t hb = (size_t)nbins * 8;
    const size_t cnt_bytes = (n_chunks + 2) * 8;
    const size_t per_start = Arena::padded(n * 8) + Arena::padded(n * 4) + Arena::padded(n) + Arena::padded(n * 32) +
                             Arena::padded(n * 4) + 3 * Arena::padded(n * 8) + Arena::padded(n * 8) + Arena::padded(n) +
                             Arena::padded(hb) + Arena::padded(ws) + Arena::padded(cnt_bytes) + 4096;
    const size_t redo = Arena::padded(chunk * V * 16) + Arena::padded(chunk * 8) + Arena::padded(chunk * 4) +
                        2 * Arena::padded(chunk) + Arena::padded(chunk * 32) + Arena::padded(chunk * 8);
    if (keep && !t_arena.reserve(per_start + Arena::padded(n * V * 16))) keep = false;   // does not fit beside the rest: chunks
    if (!keep && !t_arena.reserve(per_start + redo))
        return fail(U1GF_ENOMEM, "u1gf_pipeline_host: device allocation of %zu bytes failed", per_start + redo);
    DevBuf F, sw, stt, sg, cid, rep, mul, Frep, lam, reg, hist, wsb, gc, ids, sw2, st2, reg2, sg2, F2, cnt;
    F.take(n * 8); sw.take(n * 4); stt.take(n); sg.take(n * 32); cid.take(n * 4); rep.take(n * 8); mul.take(n * 8);
    Frep.take(n * 8); lam.take(n * 8); reg.take(n); hist.take(hb); wsb.take(ws); cnt.take(cnt_bytes);
    if (keep) {
        gc.take(n * V * 16);
    } else {
        gc.take(chunk * V * 16); ids.take(chunk * 8); sw2.take(chunk * 4); st2.take(chunk); reg2.take(chunk);
        sg2.take(chunk * 32); F2.take(chunk * 8);
    }
    int64_t* nd_dev = (int64_t*)cnt.p;
    int64_t* nin_dev = nd_dev + 1;     // one slot per u1gf_check_fp call, read back together at the end
    int launches = 0;
    DrainUnlessDone drain;
    // a2-a6 on every start, a8
    int rc = u1gf_relax_batch(o, seed, first_start, n_starts, nullptr, omega, eps, max_sweeps, check_every, (double*)F.p,
                              (int32_t*)sw.p, (uint8_t*)stt.p, (double*)sg.p, keep ? (double*)gc.p : nullptr, wsb.p, ws, nullptr);
    if (rc) return rc;
    launches += t_launches;
    rc = u1gf_count_copies(n_starts, (const double*)F.p, (const double*)sg.p, (const uint8_t*)stt.p, tol_F, tol_sig,
                           (int32_t*)cid.p, nd_dev, (int64_t*)rep.p, (int64_t*)mul.p, nbins > 0 ? (int64_t*)hist.p : nullptr,
                           nbins, wsb.p, ws, nullptr);
    if (rc) return rc;
    launches += t_launches;
    int64_t nd = 0;
    U1GF_CUDA(cudaMemcpy(&nd, nd_dev, 8, cudaMemcpyDeviceToHost));   // the one host read the path needs before it can go on
    *n_distinct_host = nd;
    o->pipeline_keep_fields = (uint64_t)nd > n_starts / 4 ? 1 : 0;
    const bool want_tables = rep_host || multiplicity_host || F_rep_host || lambda1_host || region_host;
    if (want_tables && nd > copy_capacity)     // before any copy into the caller's arrays is enqueued
        return fail(U1GF_ENOMEM, "u1gf_pipeline_host: %lld distinct copies, per-copy arrays hold %lld", (long long)nd,
                    (long long)copy_capacity);
    // per-start results: enqueued here, on the same (legacy default) stream as everything else, so they run before the
    // first-region phase, not beside it; with pinned host arrays the host goes straight on to enqueue that phase
    if (F_norm_host) U1GF_CUDA(cudaMemcpyAsync(F_norm_host, F.p, n * 8, cudaMemcpyDeviceToHost, nullptr));
    if (sweeps_host) U1GF_CUDA(cudaMemcpyAsync(sweeps_host, sw.p, n * 4, cudaMemcpyDeviceToHost, nullptr));
    if (status_host) U1GF_CUDA(cudaMemcpyAsync(status_host, stt.p, n, cudaMemcpyDeviceToHost, nullptr));
    if (sig_host) U1GF_CUDA(cudaMemcpyAsync(sig_host, sg.p, n * 32, cudaMemcpyDeviceToHost, nullptr));
    if (copy_id_host) U1GF_CUDA(cudaMemcpyAsync(copy_id_host, cid.p, n * 4, cudaMemcpyDeviceToHost, nullptr));
    if (hist_host && nbins > 0) U1GF_CUDA(cudaMemcpyAsync(hist_host, hist.p, hb, cudaMemcpyDeviceToHost, nullptr));
    // a7 on the representatives
    size_t fp_calls = 0;
    if (keep) {
        if (nd > 0) {
            rc = u1gf_check_fp(o, (uint64_t)nd, (const double*)gc.p, (const int64_t*)rep.p, tol_fp, (double*)lam.p,
                               (uint8_t*)reg.p, nin_dev, nullptr, nullptr);
            if (rc) return rc;
            launches += t_launches;
            fp_calls = 1;
        }
    } else {
        // re-relaxed with their fields written out (a start is a pure function of its index)
        for (int64_t a = 0; a < nd; a += (int64_t)chunk) {
            const uint64_t m = (uint64_t)std::min<int64_t>((int64_t)chunk, nd - a);
            add_offset_kernel<<<(unsigned)((m + 255) / 256), 256>>>(m, (const int64_t*)rep.p + a, first_start, (uint64_t*)ids.p);
            U1GF_CUDA(cudaGetLastError());
            ++launches;
            rc = u1gf_relax_batch(o, seed, 0, m, (const uint64_t*)ids.p, omega, eps, max_sweeps, check_every, (double*)F2.p,
                                  (int32_t*)sw2.p, (uint8_t*)st2.p, (double*)sg2.p, (double*)gc.p, wsb.p, ws, nullptr);
            if (rc) return rc;
            launches += t_launches;
            rc = u1gf_check_fp(o, m, (const double*)gc.p, nullptr, tol_fp, (double*)lam.p + a, (uint8_t*)reg.p + a,
                               nin_dev + fp_calls, nullptr, nullptr);
            if (rc) return rc;
            launches += t_launches;
            ++fp_calls;
        }
    }
    std::vector<int64_t> parts(fp_calls, 0);
    if (fp_calls) U1GF_CUDA(cudaMemcpyAsync(parts.data(), nin_dev, fp_calls * 8, cudaMemcpyDeviceToHost, nullptr));
    if (nd > 0) {
        if (F_rep_host) {
            gather_F_kernel<<<(unsigned)((nd + 255) / 256), 256>>>((unsigned long long)nd, (const int64_t*)rep.p, (const double*)F.p, (double*)Frep.p);
            U1GF_CUDA(cudaGetLastError());
            ++launches;
            U1GF_CUDA(cudaMemcpyAsync(F_rep_host, Frep.p, (size_t)nd * 8, cudaMemcpyDeviceToHost, nullptr));
        }
        if (rep_host) U1GF_CUDA(cudaMemcpyAsync(rep_host, rep.p, (size_t)nd * 8, cudaMemcpyDeviceToHost, nullptr));
        if (multiplicity_host) U1GF_CUDA(cudaMemcpyAsync(multiplicity_host, mul.p, (size_t)nd * 8, cudaMemcpyDeviceToHost, nullptr));
        if (lambda1_host) U1GF_CUDA(cudaMemcpyAsync(lambda1_host, lam.p, (size_t)nd * 8, cudaMemcpyDeviceToHost, nullptr));
        if (region_host) U1GF_CUDA(cudaMemcpyAsync(region_host, reg.p, (size_t)nd, cudaMemcpyDeviceToHost, nullptr));
    }
    U1GF_CUDA(cudaDeviceSynchronize());
    drain.done = true;
    int64_t n_in = 0;
    for (int64_t part : parts) n_in += part;
    *n_in_region_host = n_in;
    t_launches = launches;
    return U1GF_OK;
}

}  // extern "C"
