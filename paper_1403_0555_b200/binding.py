"""Thin ctypes binding of libu1gf.so (include/u1gf.h): same names, argument marshalling only.

torch supplies device memory and the CUDA stream; every step of the path runs in the library's kernels.
There is no CPU fallback: if the shared library is missing or no sm_100 device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libu1gf.so")

# every symbol include/u1gf.h declares: name -> (restype, argtypes)
_p = C.c_void_p
_SIGNATURES = {
    "u1gf_last_error": (C.c_char_p, []),
    "u1gf_abi_version": (C.c_int, []),
    "u1gf_create_orbit": (C.c_int, [C.c_int, _p, _p, C.POINTER(_p)]),
    "u1gf_destroy_orbit": (C.c_int, [_p]),
    "u1gf_orbit_volume": (C.c_int32, [_p]),
    "u1gf_orbit_dim": (C.c_int32, [_p]),
    "u1gf_relax_workspace_bytes": (C.c_size_t, [_p, C.c_uint64]),
    "u1gf_relax_batch": (C.c_int, [_p, C.c_uint64, C.c_uint64, C.c_uint64, _p, C.c_double, C.c_double, C.c_int32,
                                   C.c_int32, _p, _p, _p, _p, _p, _p, C.c_size_t, _p]),
    "u1gf_relax_batch_host": (C.c_int, [_p, C.c_uint64, C.c_uint64, C.c_uint64, _p, C.c_double, C.c_double,
                                        C.c_int32, C.c_int32, _p, _p, _p, _p, _p]),
    "u1gf_set_kernel": (C.c_int, [_p, C.c_int32]),
    "u1gf_kernel_name": (C.c_char_p, [_p]),
    "u1gf_check_fp": (C.c_int, [_p, C.c_uint64, _p, _p, C.c_double, _p, _p, _p, _p, _p]),
    "u1gf_check_fp_host": (C.c_int, [_p, C.c_uint64, _p, C.c_double, _p, _p, _p]),
    "u1gf_count_workspace_bytes": (C.c_size_t, [C.c_uint64]),
    "u1gf_count_copies": (C.c_int, [C.c_uint64, _p, _p, _p, C.c_double, C.c_double, _p, _p, _p, _p, _p, C.c_int32,
                                    _p, C.c_size_t, _p]),
    "u1gf_count_copies_host": (C.c_int, [C.c_uint64, _p, _p, _p, C.c_double, C.c_double, _p, _p, _p, _p, _p,
                                         C.c_int32]),
    "u1gf_discovery_curve": (C.c_int, [C.c_uint64, _p, C.c_int32, _p, _p]),
    "u1gf_paper_count_workspace_bytes": (C.c_size_t, [C.c_uint64]),
    "u1gf_paper_count": (C.c_int, [C.c_uint64, _p, _p, C.c_double, _p, _p, C.c_size_t, _p]),
    "u1gf_paper_count_static": (C.c_int, [C.c_uint64, _p, _p, C.c_double, _p, _p]),
    "u1gf_pipeline_host": (C.c_int, [_p, C.c_uint64, C.c_uint64, C.c_uint64, C.c_double, C.c_double, C.c_int32, C.c_int32,
                                     C.c_double, C.c_double, C.c_double, C.c_int32, _p, _p, _p, _p, _p, C.c_int64, _p, _p,
                                     _p, _p, _p, _p, _p, _p]),
    "u1gf_release_host_scratch": (C.c_int, []),
    "u1gf_create_ensemble": (C.c_int, [C.c_int, _p, C.c_int32, _p, _p, C.POINTER(_p)]),
    "u1gf_destroy_ensemble": (C.c_int, [_p]),
    "u1gf_ensemble_size": (C.c_int32, [_p]),
    "u1gf_ensemble_orbit": (_p, [_p, C.c_int32]),
    "u1gf_relax_ensemble_workspace_bytes": (C.c_size_t, [_p, C.c_uint64]),
    "u1gf_relax_ensemble": (C.c_int, [_p, C.c_uint64, C.c_uint64, C.c_double, C.c_double, C.c_int32, C.c_int32, _p, _p, _p,
                                      _p, _p, C.c_size_t, _p]),
    "u1gf_count_ensemble_workspace_bytes": (C.c_size_t, [C.c_uint64]),
    "u1gf_count_ensemble_onepass_workspace_bytes": (C.c_size_t, [C.c_int32, C.c_uint64]),
    "u1gf_count_copies_ensemble": (C.c_int, [C.c_int32, C.c_uint64, _p, _p, _p, C.c_double, C.c_double, _p, _p, _p, _p, _p,
                                             C.c_int32, _p, C.c_size_t, _p]),
    "u1gf_ensemble_stats": (C.c_int, [C.c_int32, C.c_uint64, _p, _p, _p, _p, _p, _p, _p]),
    "u1gf_relative_deviation_hist": (C.c_int, [C.c_int32, C.c_uint64, _p, _p, _p, _p, _p, C.c_double, C.c_int32, _p, _p, _p,
                                               _p, _p]),
    "u1gf_hist_ratio": (C.c_int, [C.c_int32, _p, _p, _p, _p, _p]),
    "u1gf_merge_workspace_bytes": (C.c_size_t, [C.c_uint64]),
    "u1gf_merge_copy_tables": (C.c_int, [C.c_uint64, _p, _p, _p, _p, C.c_double, C.c_double, _p, _p, _p, _p, _p,
                                         C.c_size_t, _p]),
}

# include/u1gf_measure.h: one symbol of libu1gf.so and the probes of libu1gf_measure.so
_MEASURE_SIGNATURES_MAIN = {"u1gf_last_launch_count": (C.c_int32, [])}
_MEASURE_SIGNATURES = {
    "u1gf_measure_last_error": (C.c_char_p, []),
    "u1gf_measure_fp64_peak": (C.c_int, [C.c_double, C.POINTER(C.c_double), _p]),
    "u1gf_measure_fp64_rate": (C.c_int, [C.c_int32, C.c_double, C.POINTER(C.c_double), _p]),
    "u1gf_measure_smem_peak": (C.c_int, [C.c_double, C.POINTER(C.c_double), _p]),
    "u1gf_measure_smem_rate": (C.c_int, [C.c_int32, C.c_double, C.POINTER(C.c_double), _p]),
    "u1gf_measure_dsmem_rate": (C.c_int, [C.c_int32, C.c_int32, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_int32), _p]),
}
MEASURE_LIB_PATH = os.path.join(_HERE, "libu1gf_measure.so")

_lib = None
_mlib = None


class U1gfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libu1gf error {code}: {msg}")
        self.code = code


def lib():
    """Load libu1gf.so (fails loudly if it was not built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not built; run `python -m paper_1403_0555_b200.build`")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in {**_SIGNATURES, **_MEASURE_SIGNATURES_MAIN}.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def use_library(path):
    """Load another build of the method library (tests: build.build_variant) in place of libu1gf.so."""
    global _lib, LIB_PATH
    LIB_PATH = path
    _lib = None
    return lib()


def measure_lib():
    """Load libu1gf_measure.so (include/u1gf_measure.h: roofline probes, not the method)."""
    global _mlib
    if _mlib is None:
        if not os.path.exists(MEASURE_LIB_PATH):
            raise FileNotFoundError(f"{MEASURE_LIB_PATH} not built; run `python -m paper_1403_0555_b200.build`")
        L = C.CDLL(MEASURE_LIB_PATH)
        for name, (res, args) in _MEASURE_SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _mlib = L
    return _mlib


def exported_symbols():
    return sorted(_SIGNATURES)


def measure_symbols():
    return sorted({**_MEASURE_SIGNATURES_MAIN, **_MEASURE_SIGNATURES})


def _check(rc):
    if rc != 0:
        raise U1gfError(rc, lib().u1gf_last_error().decode())


def _np_ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dev_ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Orbit:
    """u1gf_create_orbit / u1gf_destroy_orbit (a1)."""

    def __init__(self, extents, theta):
        e = np.ascontiguousarray(extents, dtype=np.int32)
        t = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1)
        if t.size != int(np.prod(e)) * e.size:
            raise ValueError("theta must have V*d entries (index i*d+mu)")
        h = C.c_void_p()
        _check(lib().u1gf_create_orbit(int(e.size), _np_ptr(e), _np_ptr(t), C.byref(h)))
        self.handle = h
        self.extents = tuple(int(x) for x in e)
        self.d = int(e.size)
        self.V = int(np.prod(e))

    def close(self):
        if getattr(self, "_borrowed", False):   # a member of an Ensemble: the ensemble frees it
            self.handle = None
            return
        if getattr(self, "handle", None):
            lib().u1gf_destroy_orbit(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:   # interpreter shutdown: module globals may already be gone
            pass

    def set_kernel(self, which: int):
        _check(lib().u1gf_set_kernel(self.handle, int(which)))

    @property
    def kernel_name(self) -> str:
        return lib().u1gf_kernel_name(self.handle).decode()


class Ensemble:
    """u1gf_ensemble handle: n_orbits orbits of one lattice shape relaxed in one launch."""

    def __init__(self, extents, thetas, seeds):
        ext = np.ascontiguousarray(extents, dtype=np.int32)
        th = np.ascontiguousarray(thetas, dtype=np.float64)
        sd = np.ascontiguousarray(seeds, dtype=np.uint64)
        self.extents = tuple(int(e) for e in ext)
        self.d, self.V, self.n_orbits = ext.size, int(np.prod(ext)), int(sd.size)
        assert th.size == self.n_orbits * self.V * self.d, "thetas must be [n_orbits][V*d]"
        h = C.c_void_p()
        _check(lib().u1gf_create_ensemble(self.d, _np_ptr(ext), self.n_orbits, _np_ptr(th), _np_ptr(sd), C.byref(h)))
        self.handle = h
        self.seeds = sd

    def orbit(self, k):
        """Member k as an Orbit (borrowed: the ensemble owns it)."""
        o = Orbit.__new__(Orbit)
        o.extents, o.d, o.V = self.extents, self.d, self.V
        o.handle = C.c_void_p(lib().u1gf_ensemble_orbit(self.handle, int(k)))
        o._borrowed = True
        return o

    def close(self):
        if getattr(self, "handle", None):
            _check(lib().u1gf_destroy_ensemble(self.handle))
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def relax_ensemble(ens: Ensemble, n_starts_per_orbit, *, first_start=0, omega=1.7, eps=1e-13, max_sweeps=20000,
                   check_every=1, workspace=None):
    """u1gf_relax_ensemble -> dict of device tensors shaped [n_orbits, n] (sig [n_orbits, n, 4])."""
    import torch
    n, no = int(n_starts_per_orbit), ens.n_orbits
    out = dict(F_norm=torch.empty((no, n), dtype=torch.float64, device="cuda"),
               sweeps=torch.empty((no, n), dtype=torch.int32, device="cuda"),
               status=torch.empty((no, n), dtype=torch.uint8, device="cuda"),
               sig=torch.empty((no, n, 4), dtype=torch.float64, device="cuda"))
    need = lib().u1gf_relax_ensemble_workspace_bytes(ens.handle, n)
    if workspace is None or workspace.numel() < need + 256:
        workspace = _workspace(need)
    out["workspace"] = workspace
    _check(lib().u1gf_relax_ensemble(ens.handle, int(first_start), n, float(omega), float(eps), int(max_sweeps),
                                     int(check_every), _dev_ptr(out["F_norm"]), _dev_ptr(out["sweeps"]),
                                     _dev_ptr(out["status"]), _dev_ptr(out["sig"]), _aligned_ptr(workspace), need, _stream()))
    return out


def count_copies_ensemble(F_norm, sig, status, tol_F=1e-10, tol_sig=1e-4, nbins=0, workspace=None, one_pass=True):
    """u1gf_count_copies_ensemble on [n_orbits, n] device tensors -> per-orbit tables ([n_orbits, n], n_distinct [n_orbits]).
    one_pass: give the call the larger workspace with which it de-duplicates all orbits in one pass (where available)."""
    import torch
    no, n = int(F_norm.shape[0]), int(F_norm.shape[1])
    copy_id = torch.empty((no, n), dtype=torch.int32, device="cuda")
    nd = torch.zeros(no, dtype=torch.int64, device="cuda")
    rep = torch.empty((no, max(n, 1)), dtype=torch.int64, device="cuda")
    mult = torch.empty((no, max(n, 1)), dtype=torch.int64, device="cuda")
    hist = torch.empty((no, nbins), dtype=torch.int64, device="cuda") if nbins else None
    need = lib().u1gf_count_ensemble_workspace_bytes(n)
    if one_pass:
        need = max(need, lib().u1gf_count_ensemble_onepass_workspace_bytes(no, n))
    if workspace is None or workspace.numel() < need + 256:
        workspace = _workspace(need)
    _check(lib().u1gf_count_copies_ensemble(no, n, _dev_ptr(F_norm), _dev_ptr(sig), _dev_ptr(status), float(tol_F),
                                            float(tol_sig), _dev_ptr(copy_id), _dev_ptr(nd), _dev_ptr(rep), _dev_ptr(mult),
                                            _dev_ptr(hist), int(nbins), _aligned_ptr(workspace), need, _stream()))
    return dict(copy_id=copy_id, n_distinct=nd, rep=rep, multiplicity=mult, hist=hist, workspace=workspace)


def merge_copy_tables(F_rep, sig_rep, first_start, multiplicity, tol_F=1e-10, tol_sig=1e-4):
    """u1gf_merge_copy_tables on device tensors -> dict(merged_id, n_merged, first_start, multiplicity)."""
    import torch
    m = int(F_rep.numel())
    mid = torch.empty(m, dtype=torch.int32, device="cuda")
    nm = torch.zeros(1, dtype=torch.int64, device="cuda")
    mfs = torch.empty(max(m, 1), dtype=torch.int64, device="cuda")
    mmu = torch.empty(max(m, 1), dtype=torch.int64, device="cuda")
    need = lib().u1gf_merge_workspace_bytes(m)
    ws = _workspace(need)
    _check(lib().u1gf_merge_copy_tables(m, _dev_ptr(F_rep.contiguous()), _dev_ptr(sig_rep.contiguous()),
                                        _dev_ptr(first_start.contiguous()), _dev_ptr(multiplicity.contiguous()),
                                        float(tol_F), float(tol_sig), _dev_ptr(mid), _dev_ptr(nm), _dev_ptr(mfs),
                                        _dev_ptr(mmu), _aligned_ptr(ws), need, _stream()))
    return dict(merged_id=mid, n_merged=nm, first_start=mfs, multiplicity=mmu)


def ensemble_stats(n_orbits, n_per_orbit, F_norm, rep, n_distinct, n_in_region=None):
    """u1gf_ensemble_stats on the device arrays of relax_ensemble / count_copies_ensemble -> dict(best_x [n_orbits], stats [8])."""
    import torch
    best = torch.empty(int(n_orbits), dtype=torch.float64, device="cuda")
    stats = torch.empty(8, dtype=torch.float64, device="cuda")
    _check(lib().u1gf_ensemble_stats(int(n_orbits), int(n_per_orbit), _dev_ptr(F_norm), _dev_ptr(rep), _dev_ptr(n_distinct),
                                     _dev_ptr(n_in_region), _dev_ptr(best), _dev_ptr(stats), _stream()))
    return dict(best_x=best, stats=stats)


def relative_deviation_hist(n_orbits, n_per_orbit, F_norm, rep, multiplicity, n_distinct, best_x, dev_max, nbins):
    """u1gf_relative_deviation_hist -> dict(counts [n_orbits, nbins], n_converged [n_orbits], avg [nbins], n_orbits_used [1])."""
    import torch
    counts = torch.empty((int(n_orbits), int(nbins)), dtype=torch.int64, device="cuda")
    nconv = torch.empty(int(n_orbits), dtype=torch.int64, device="cuda")
    avg = torch.empty(int(nbins), dtype=torch.float64, device="cuda")
    used = torch.empty(1, dtype=torch.int64, device="cuda")
    _check(lib().u1gf_relative_deviation_hist(int(n_orbits), int(n_per_orbit), _dev_ptr(F_norm), _dev_ptr(rep),
                                              _dev_ptr(multiplicity), _dev_ptr(n_distinct), _dev_ptr(best_x), float(dev_max),
                                              int(nbins), _dev_ptr(counts), _dev_ptr(nconv), _dev_ptr(avg), _dev_ptr(used),
                                              _stream()))
    return dict(counts=counts, n_converged=nconv, avg=avg, n_orbits_used=used)


def hist_ratio(hist_small, hist_big):
    """u1gf_hist_ratio on two device int64 histograms -> dict(ratio [nbins], n_only [2])."""
    import torch
    nb = int(hist_small.numel())
    assert int(hist_big.numel()) == nb
    ratio = torch.empty(nb, dtype=torch.float64, device="cuda")
    n_only = torch.empty(2, dtype=torch.int64, device="cuda")
    _check(lib().u1gf_hist_ratio(nb, _dev_ptr(hist_small), _dev_ptr(hist_big), _dev_ptr(ratio), _dev_ptr(n_only), _stream()))
    return dict(ratio=ratio, n_only=n_only)


def pipeline_host(orbit, seed, n_starts, *, first_start=0, omega=1.7, eps=1e-13, max_sweeps=20000, check_every=1,
                  tol_F=1e-10, tol_sig=1e-4, tol_fp=1e-8, nbins=0, out=None, copy_capacity=None):
    """u1gf_pipeline_host: the whole hot path with host (numpy) result arrays.  `out` = host_buffers(n) reuses pinned
    arrays; per-copy arrays hold `copy_capacity` entries (default n)."""
    n = int(n_starts)
    cap = n if copy_capacity is None else int(copy_capacity)
    if out is None:
        out = host_buffers(n, pinned=False)
    per_copy = out.get("per_copy")
    if per_copy is None or per_copy["lambda1"].size < cap:
        per_copy = dict(F_rep=np.zeros(max(cap, 1)), lambda1=np.zeros(max(cap, 1)),
                        region=np.zeros(max(cap, 1), dtype=np.uint8))
        out["per_copy"] = per_copy
    hist = np.zeros(nbins, dtype=np.int64) if nbins else None
    nd, nin = np.zeros(1, dtype=np.int64), np.zeros(1, dtype=np.int64)
    _check(lib().u1gf_pipeline_host(orbit.handle, int(seed), int(first_start), n, float(omega), float(eps), int(max_sweeps),
                                    int(check_every), float(tol_F), float(tol_sig), float(tol_fp), int(nbins),
                                    _np_ptr(out["F_norm"]), _np_ptr(out["sweeps"]), _np_ptr(out["status"]),
                                    _np_ptr(out["sig"]), _np_ptr(out["copy_id"]), cap, _np_ptr(nd), _np_ptr(out["rep"]),
                                    _np_ptr(out["multiplicity"]), _np_ptr(per_copy["F_rep"]), _np_ptr(per_copy["lambda1"]),
                                    _np_ptr(per_copy["region"]), _np_ptr(nin), _np_ptr(hist)))
    k = int(nd[0])
    return dict(F_norm=out["F_norm"], sweeps=out["sweeps"], status=out["status"], sig=out["sig"], copy_id=out["copy_id"],
                n_distinct=k, rep=out["rep"][:k], multiplicity=out["multiplicity"][:k], F_rep=per_copy["F_rep"][:k],
                lambda1=per_copy["lambda1"][:k], region=per_copy["region"][:k], n_in_region=int(nin[0]), hist=hist)


def _workspace(nbytes):
    import torch
    return torch.empty(max(int(nbytes), 256) + 256, dtype=torch.uint8, device="cuda")


def _aligned_ptr(ws):
    p = ws.data_ptr()
    return C.c_void_p((p + 255) & ~255)


def relax_batch(orbit: Orbit, seed, n_starts, *, first_start=0, start_ids=None, omega=1.7, eps=1e-13,
                max_sweeps=20000, check_every=1, want_g=False, out=None, workspace=None):
    """u1gf_relax_batch with device (torch) result tensors.  Returns a dict of torch tensors on the GPU.
    `out` / `workspace` may carry preallocated tensors from a previous call (nothing is then allocated)."""
    import torch
    if start_ids is not None:
        if not isinstance(start_ids, torch.Tensor):
            start_ids = torch.as_tensor(np.ascontiguousarray(start_ids, dtype=np.uint64).view(np.int64), device="cuda")
        n_starts = start_ids.numel()
    n = int(n_starts)
    if out is None:
        out = dict(F_norm=torch.empty(n, dtype=torch.float64, device="cuda"),
                   sweeps=torch.empty(n, dtype=torch.int32, device="cuda"),
                   status=torch.empty(n, dtype=torch.uint8, device="cuda"),
                   sig=torch.empty((n, 4), dtype=torch.float64, device="cuda"),
                   g_canon=torch.empty((n, orbit.V, 2), dtype=torch.float64, device="cuda") if want_g else None)
    need = lib().u1gf_relax_workspace_bytes(orbit.handle, n)
    if workspace is None or workspace.numel() < need + 256:
        workspace = _workspace(need)
    out["workspace"] = workspace
    _check(lib().u1gf_relax_batch(orbit.handle, int(seed), int(first_start), n, _dev_ptr(start_ids), float(omega),
                                  float(eps), int(max_sweeps), int(check_every), _dev_ptr(out["F_norm"]),
                                  _dev_ptr(out["sweeps"]), _dev_ptr(out["status"]), _dev_ptr(out["sig"]),
                                  _dev_ptr(out.get("g_canon")), _aligned_ptr(workspace), need, _stream()))
    return out


def host_buffers(n, V=0, want_g=False, pinned=True):
    """Result arrays for the *_host calls (F_norm, sweeps, status, sig, copy_id, rep, multiplicity[, g_canon]) in
    page-locked host memory (numpy views of pinned torch tensors), so that the library's device<->host copies run at
    PCIe speed and a caller can reuse them across calls instead of faulting in fresh pages every time."""
    import torch

    def arr(shape, dtype):
        return torch.empty(shape, dtype=dtype, pin_memory=pinned).numpy()
    n = int(n)
    return dict(F_norm=arr(n, torch.float64), sweeps=arr(n, torch.int32), status=arr(n, torch.uint8),
                sig=arr((n, 4), torch.float64), copy_id=arr(n, torch.int32), rep=arr(max(n, 1), torch.int64),
                multiplicity=arr(max(n, 1), torch.int64),
                g_canon=arr((n, int(V), 2), torch.float64) if want_g else None)


def relax_batch_host(orbit: Orbit, seed, n_starts, *, first_start=0, start_ids=None, omega=1.7, eps=1e-13,
                     max_sweeps=20000, check_every=1, want_g=False, out=None):
    """u1gf_relax_batch_host: numpy result arrays, device<->host copies inside the call.  `out` (host_buffers())
    supplies the result arrays; otherwise fresh pageable ones are made."""
    ids = None
    if start_ids is not None:
        ids = np.ascontiguousarray(start_ids, dtype=np.uint64)
        n_starts = ids.size
    n = int(n_starts)
    if out is None:
        out = dict(F_norm=np.zeros(n), sweeps=np.zeros(n, dtype=np.int32), status=np.zeros(n, dtype=np.uint8),
                   sig=np.zeros((n, 4)), g_canon=np.zeros((n, orbit.V, 2)) if want_g else None)
    elif out["F_norm"].size != n or (want_g and out.get("g_canon") is None):
        raise ValueError("relax_batch_host: `out` buffers do not match n_starts / want_g")
    _check(lib().u1gf_relax_batch_host(orbit.handle, int(seed), int(first_start), n, _np_ptr(ids), float(omega),
                                       float(eps), int(max_sweeps), int(check_every), _np_ptr(out["F_norm"]),
                                       _np_ptr(out["sweeps"]), _np_ptr(out["status"]), _np_ptr(out["sig"]),
                                       _np_ptr(out["g_canon"])))
    return out


def check_fp(orbit: Orbit, g, tol_fp=1e-8, want_steps=False, index=None):
    """u1gf_check_fp on a device tensor g[., V, 2] -> dict(lambda1, region, n_in_region) of device tensors.  `index`
    (device int64 tensor) selects the configurations g[index[k]]; without it all of g is tested."""
    import torch
    g = g.contiguous()
    n = int(g.shape[0]) if g.numel() else 0
    if index is not None:
        index = index.contiguous()
        n = int(index.numel())
    lam = torch.empty(n, dtype=torch.float64, device="cuda")
    reg = torch.empty(n, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    steps = torch.empty(n, dtype=torch.int32, device="cuda") if want_steps else None
    _check(lib().u1gf_check_fp(orbit.handle, n, _dev_ptr(g), _dev_ptr(index), float(tol_fp), _dev_ptr(lam), _dev_ptr(reg),
                               _dev_ptr(cnt), _dev_ptr(steps), _stream()))
    return dict(lambda1=lam, region=reg, n_in_region=cnt, steps=steps)


def check_fp_host(orbit: Orbit, g, tol_fp=1e-8):
    g = np.ascontiguousarray(g, dtype=np.float64).reshape(-1, orbit.V, 2)
    n = g.shape[0]
    lam = np.zeros(n)
    reg = np.zeros(n, dtype=np.uint8)
    cnt = np.zeros(1, dtype=np.int64)
    _check(lib().u1gf_check_fp_host(orbit.handle, n, _np_ptr(g), float(tol_fp), _np_ptr(lam), _np_ptr(reg),
                                    _np_ptr(cnt)))
    return dict(lambda1=lam, region=reg, n_in_region=int(cnt[0]))


def count_copies(F_norm, sig, status, tol_F=1e-10, tol_sig=1e-4, nbins=0, workspace=None):
    """u1gf_count_copies on device tensors -> dict of device tensors (copy_id, n_distinct, rep, multiplicity, hist).
    rep / multiplicity are full-length; entries beyond n_distinct are undefined."""
    import torch
    n = int(F_norm.numel())
    copy_id = torch.empty(n, dtype=torch.int32, device="cuda")
    nd = torch.zeros(1, dtype=torch.int64, device="cuda")
    rep = torch.empty(max(n, 1), dtype=torch.int64, device="cuda")
    mult = torch.empty(max(n, 1), dtype=torch.int64, device="cuda")
    hist = torch.empty(nbins, dtype=torch.int64, device="cuda") if nbins else None
    need = lib().u1gf_count_workspace_bytes(n)
    if workspace is None or workspace.numel() < need + 256:
        workspace = _workspace(need)
    _check(lib().u1gf_count_copies(n, _dev_ptr(F_norm), _dev_ptr(sig), _dev_ptr(status), float(tol_F), float(tol_sig),
                                   _dev_ptr(copy_id), _dev_ptr(nd), _dev_ptr(rep), _dev_ptr(mult), _dev_ptr(hist),
                                   int(nbins), _aligned_ptr(workspace), need, _stream()))
    return dict(copy_id=copy_id, n_distinct=nd, rep=rep, multiplicity=mult, hist=hist, workspace=workspace)


def count_copies_host(F_norm, sig, status, tol_F=1e-10, tol_sig=1e-4, nbins=0, out=None):
    F = np.ascontiguousarray(F_norm, dtype=np.float64)
    S = np.ascontiguousarray(sig, dtype=np.float64).reshape(-1, 4)
    st = np.ascontiguousarray(status, dtype=np.uint8)
    n = F.size
    nd = np.zeros(1, dtype=np.int64)
    if out is not None and out["copy_id"].size == n:
        copy_id, rep, mult = out["copy_id"], out["rep"], out["multiplicity"]
    else:
        copy_id = np.zeros(n, dtype=np.int32)
        rep = np.zeros(max(n, 1), dtype=np.int64)
        mult = np.zeros(max(n, 1), dtype=np.int64)
    hist = np.zeros(nbins, dtype=np.int64) if nbins else None
    _check(lib().u1gf_count_copies_host(n, _np_ptr(F), _np_ptr(S), _np_ptr(st), float(tol_F), float(tol_sig),
                                        _np_ptr(copy_id), _np_ptr(nd), _np_ptr(rep), _np_ptr(mult), _np_ptr(hist),
                                        int(nbins)))
    k = int(nd[0])
    return dict(copy_id=copy_id, n_distinct=k, rep=rep[:k], multiplicity=mult[:k], hist=hist)


def discovery_curve(rep, n_distinct: int, n_levels: int):
    """u1gf_discovery_curve: rep = device int64 tensor from count_copies -> device int64 tensor [n_levels]."""
    import torch
    curve = torch.empty(int(n_levels), dtype=torch.int64, device="cuda")
    _check(lib().u1gf_discovery_curve(int(n_distinct), _dev_ptr(rep), int(n_levels), _dev_ptr(curve), _stream()))
    return curve


def paper_count(F_norm, status, scale=1e8, workspace=None):
    """u1gf_paper_count on device tensors -> device int64 tensor [1]."""
    import torch
    n = int(F_norm.numel())
    nk = torch.zeros(1, dtype=torch.int64, device="cuda")
    need = lib().u1gf_paper_count_workspace_bytes(n)
    if workspace is None or workspace.numel() < need + 256:
        workspace = _workspace(need)
    _check(lib().u1gf_paper_count(n, _dev_ptr(F_norm), _dev_ptr(status), float(scale), _dev_ptr(nk),
                                  _aligned_ptr(workspace), need, _stream()))
    return nk


PAPER_COUNT_STATIC_MAX_N = 1 << 20   # U1GF_PAPER_COUNT_STATIC_MAX_N of include/u1gf.h


def paper_count_static(F_norm, status, scale=1e8, out=None):
    """u1gf_paper_count_static: the count of u1gf_paper_count for callers that cannot get device memory (all of it handed
    out by their host application, no allocator to ask, or an allocation stall they cannot afford): the scratch is a
    32 MiB array built into the library, so nothing is allocated here either when `out` (device int64 [1]) is given.
    At most PAPER_COUNT_STATIC_MAX_N records; every call shares the one array, so calls must not overlap on the GPU.
    The first call on a device does the set-up (include/u1gf.h) -- make it before any stream capture."""
    n = int(F_norm.numel())
    if out is None:
        import torch
        out = torch.empty(1, dtype=torch.int64, device="cuda")
    _check(lib().u1gf_paper_count_static(n, _dev_ptr(F_norm), _dev_ptr(status), float(scale), _dev_ptr(out), _stream()))
    return out


def _mcheck(rc):
    if rc != 0:
        raise U1gfError(rc, measure_lib().u1gf_measure_last_error().decode())


def measure_fp64_peak(ms=200.0) -> float:
    v = C.c_double(0)
    _mcheck(measure_lib().u1gf_measure_fp64_peak(float(ms), C.byref(v), _stream()))
    return v.value


def measure_fp64_rate(pattern: int, ms=200.0) -> float:
    v = C.c_double(0)
    _mcheck(measure_lib().u1gf_measure_fp64_rate(int(pattern), float(ms), C.byref(v), _stream()))
    return v.value


def measure_smem_peak(ms=200.0) -> float:
    v = C.c_double(0)
    _mcheck(measure_lib().u1gf_measure_smem_peak(float(ms), C.byref(v), _stream()))
    return v.value


def measure_smem_rate(mix: int, ms=200.0) -> float:
    v = C.c_double(0)
    _mcheck(measure_lib().u1gf_measure_smem_rate(int(mix), float(ms), C.byref(v), _stream()))
    return v.value


def measure_dsmem_rate(cluster_size: int, remote: bool, ms=100.0):
    """-> (bytes per second and SM, clusters of that size resident at once)."""
    v, n = C.c_double(0), C.c_int32(0)
    _mcheck(measure_lib().u1gf_measure_dsmem_rate(int(cluster_size), 1 if remote else 0, float(ms), C.byref(v), C.byref(n),
                                                  _stream()))
    return v.value, n.value


def last_launch_count() -> int:
    return int(lib().u1gf_last_launch_count())
