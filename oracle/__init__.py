"""CPU oracle for the u1gf hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_1403_0555_b200 (the CUDA path) and imports nothing from it.

Two parts:
  * u1gf_oracle.cpp (plain C++17, FP64, scalar loops): links O1, starts O2, sweeps O3, stop rule O4,
    functional O5, canonical form + signature O6, dense Faddeev-Popov matrix O7.  Called via ctypes.
  * this file (numpy): lowest non-trivial FP eigenvalue O7 (LAPACK `eigvalsh` as the library step),
    copy identity / de-duplication / counting O8-O9 written out step by step.

Every function cites PAPER.md lines (section / equation) or a DESIGN.md reading R<k>.
Pins: tests/test_oracle_*.py.  Unpinned by construction: which copy a given (seed, start) falls into.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        p = C.c_void_p
        L.u1gf_oracle_philox4x32_10.argtypes = [p, p, p]
        L.u1gf_oracle_philox4x32_10.restype = None
        L.u1gf_oracle_links.argtypes = [C.c_int, p, p, p]
        L.u1gf_oracle_start.argtypes = [C.c_int, C.c_uint64, C.c_uint64, p]
        L.u1gf_oracle_sweeps.argtypes = [C.c_int, p, p, p, C.c_double, C.c_int32, p]
        L.u1gf_oracle_measure.argtypes = [C.c_int, p, p, p, p, p, p]
        L.u1gf_oracle_neighbour_sums.argtypes = [C.c_int, p, p, p, p]
        L.u1gf_oracle_canonicalise.argtypes = [C.c_int, p, p, p]
        L.u1gf_oracle_signature_signs.argtypes = [C.c_int, p, p]
        L.u1gf_oracle_relax.argtypes = [C.c_int, p, p, C.c_uint64, C.c_uint64, C.c_uint64, p, C.c_double,
                                        C.c_double, C.c_int32, C.c_int32, p, p, p, p, p, p, p, C.c_int32]
        L.u1gf_oracle_fp_matrix.argtypes = [C.c_int, p, p, p, p]
        L.u1gf_oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _ext(extents):
    e = np.ascontiguousarray(extents, dtype=np.int32)
    assert 1 <= e.size <= 4 and (e >= 2).all(), "extents: 1..4 directions, each >= 2"
    return e


def _theta(extents, theta):
    e = _ext(extents)
    t = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1)
    assert t.size == int(np.prod(e)) * e.size, "theta must have V*d entries, index i*d+mu"
    return e, t


def num_threads() -> int:
    return int(lib().u1gf_oracle_num_threads())


def philox4x32_10(ctr, key):
    """Raw Philox4x32-10 block (ref [59])."""
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().u1gf_oracle_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def links(extents, theta):
    """O1: U[V,d,2] = (cos theta, sin theta)."""
    e, t = _theta(extents, theta)
    U = np.zeros(t.size * 2)
    assert lib().u1gf_oracle_links(e.size, _ptr(e), _ptr(t), _ptr(U)) == 0
    return U.reshape(-1, e.size, 2)


def start(V, seed, s):
    """O2: random start s as g[V,2]."""
    g = np.zeros((V, 2))
    assert lib().u1gf_oracle_start(int(V), int(seed), int(s), _ptr(g)) == 0
    return g


def sweeps(extents, theta, g, omega, n_sweeps=1):
    """O3: n_sweeps full checkerboard sweeps on a copy of g (Eq. 4-5; R2, R3).
    Returns (g_new, skipped)."""
    e, t = _theta(extents, theta)
    g2 = np.array(g, dtype=np.float64, order="C", copy=True)
    sk = C.c_int32(0)
    assert lib().u1gf_oracle_sweeps(e.size, _ptr(e), _ptr(t), _ptr(g2), float(omega), int(n_sweeps), C.byref(sk)) == 0
    return g2, bool(sk.value)


def measure(extents, theta, g):
    """O4/O5: returns (F, vartheta, Delta[V]) on the field g (Eq. 3; L38; L133/R5)."""
    e, t = _theta(extents, theta)
    g2 = np.ascontiguousarray(g, dtype=np.float64)
    V = int(np.prod(e))
    F = C.c_double(0)
    vt = C.c_double(0)
    D = np.zeros(V)
    assert lib().u1gf_oracle_measure(e.size, _ptr(e), _ptr(t), _ptr(g2), C.byref(F), C.byref(vt), _ptr(D)) == 0
    return F.value, vt.value, D


def neighbour_sums(extents, theta, g):
    """w_i = conj(K_i) of Eq. 5 for every site, as [V,2]."""
    e, t = _theta(extents, theta)
    g2 = np.ascontiguousarray(g, dtype=np.float64)
    w = np.zeros((int(np.prod(e)), 2))
    assert lib().u1gf_oracle_neighbour_sums(e.size, _ptr(e), _ptr(t), _ptr(g2), _ptr(w)) == 0
    return w


def canonicalise(g):
    """O6: (g_canon[V,2], sig[4]); angle at the last site fixed to zero."""
    g2 = np.ascontiguousarray(g, dtype=np.float64).reshape(-1, 2)
    gc = np.zeros_like(g2)
    sig = np.zeros(4)
    assert lib().u1gf_oracle_canonicalise(g2.shape[0], _ptr(g2), _ptr(gc), _ptr(sig)) == 0
    return gc, sig


def signature_signs(V):
    a = np.zeros((4, V))
    b = np.zeros((4, V))
    lib().u1gf_oracle_signature_signs(int(V), _ptr(a), _ptr(b))
    return a, b


def relax(extents, theta, seed, n_starts, *, first_start=0, start_ids=None, omega=1.7, eps=1e-13,
          max_sweeps=20000, check_every=1, want_g=False, n_threads=0):
    """O2-O6 for a batch of starts.  Returns a dict of per-start arrays (see u1gf_oracle_relax)."""
    e, t = _theta(extents, theta)
    V = int(np.prod(e))
    ids = None
    if start_ids is not None:
        ids = np.ascontiguousarray(start_ids, dtype=np.uint64)
        n_starts = ids.size
    n = int(n_starts)
    out = dict(F_norm=np.zeros(n), sweeps=np.zeros(n, dtype=np.int32), status=np.zeros(n, dtype=np.uint8),
               sig=np.zeros((n, 4)), g_canon=np.zeros((n, V, 2)) if want_g else None,
               vt_stop=np.zeros(n), vt_prev=np.zeros(n))
    rc = lib().u1gf_oracle_relax(e.size, _ptr(e), _ptr(t), int(seed), int(first_start), n, _ptr(ids), float(omega),
                                 float(eps), int(max_sweeps), int(check_every), _ptr(out["F_norm"]),
                                 _ptr(out["sweeps"]), _ptr(out["status"]), _ptr(out["sig"]), _ptr(out["g_canon"]),
                                 _ptr(out["vt_stop"]), _ptr(out["vt_prev"]), int(n_threads))
    assert rc == 0, "u1gf_oracle_relax: invalid arguments"
    return out


# ------------------------------------------------------------------------------------------------
# O7: first-Gribov-region test (readings R9)
# ------------------------------------------------------------------------------------------------
def fp_matrix(extents, theta, g):
    """Dense FP operator M[V,V] = Hessian of -F w.r.t. the gauge angles at g."""
    e, t = _theta(extents, theta)
    g2 = np.ascontiguousarray(g, dtype=np.float64)
    V = int(np.prod(e))
    M = np.zeros((V, V))
    assert lib().u1gf_oracle_fp_matrix(e.size, _ptr(e), _ptr(t), _ptr(g2), _ptr(M)) == 0
    return M


def fp_lambda1(extents, theta, g, tol_fp=1e-8):
    """lambda_1 = smallest eigenvalue of M on the orthogonal complement of the constant vector.

    M 1 = 0 exactly (global gauge freedom), M is symmetric, so its other eigenvectors lie in
    1-perp; adding c * (1 1^T)/V with c = 4d+1 > lambda_max (Gershgorin: lambda_max <= 4d) moves the zero
    mode to c and leaves the rest untouched, hence lambda_1 = min eig(M + c 11^T/V).
    region: 1 if lambda_1 > tol_fp (inside), 2 if |lambda_1| <= tol_fp (marginal, "semi"definite L9),
    0 if lambda_1 < -tol_fp (outside the first Gribov region).
    """
    M = fp_matrix(extents, theta, g)
    V = M.shape[0]
    d = len(_ext(extents))
    c = 4.0 * d + 1.0
    lam = float(np.linalg.eigvalsh(M + (c / V) * np.ones((V, V)))[0])
    region = 1 if lam > tol_fp else (2 if abs(lam) <= tol_fp else 0)
    return lam, region


# ------------------------------------------------------------------------------------------------
# O8/O9: copy identity, de-duplication, counting (readings R7, R8, R15)
# ------------------------------------------------------------------------------------------------
def count_copies(F_norm, sig, status, tol_F=1e-10, tol_sig=1e-4, nbins=0, g_canon=None, tol_g=5e-2):
    """Step-by-step de-duplication of converged starts.

    1. keep records with status bit0 clear (converged); the others get copy_id = -1;
    2. sort the kept records by F/(dV) (ties by position) -- the paper sorts its functional values (L129);
    3. cut the sorted list into maximal runs whose adjacent gaps are <= tol_F;
    4. inside a run, repeatedly take the unassigned member with the smallest position as leader and attach
       to it every unassigned member whose signature agrees with the leader's within tol_sig (max-norm);
    5. number the copies in order of first discovery = increasing leader position (L149: counts are read
       off as a function of the number of samples);
    6. per copy: representative = leader (R8), multiplicity; histogram of the representative's F/(dV)
       weighted by multiplicity, nbins equal bins on [0,1] (L167 uses width 1e-4; R15).
    If g_canon is given the full-configuration test max_i |g~_i - g~'_i| <= tol_g must reproduce the same
    partition (asserted), and its margins are reported.
    """
    F = np.asarray(F_norm, dtype=np.float64)
    S = np.asarray(sig, dtype=np.float64).reshape(-1, 4)
    st = np.asarray(status, dtype=np.uint8)
    n = F.size
    copy_id = np.full(n, -1, dtype=np.int32)
    leader_of = np.full(n, -1, dtype=np.int64)
    keep = np.nonzero((st & 1) == 0)[0]
    order = keep[np.argsort(F[keep], kind="stable")]
    leaders = []
    margins = dict(max_within_F=0.0, max_within_sig=0.0, min_between_sig=np.inf, min_run_gap_F=np.inf,
                   max_within_g=0.0, min_between_g=np.inf)
    if order.size:
        gaps = np.diff(F[order])
        cuts = np.nonzero(gaps > tol_F)[0]
        if cuts.size:
            margins["min_run_gap_F"] = float(gaps[cuts].min())
        bounds = np.concatenate(([0], cuts + 1, [order.size]))
        for r in range(bounds.size - 1):
            run = np.sort(order[bounds[r]:bounds[r + 1]])
            if run.size == 1:
                leader_of[run[0]] = run[0]
                leaders.append(int(run[0]))
                continue
            unassigned = np.ones(run.size, dtype=bool)
            run_leaders = []
            while unassigned.any():
                lead = run[np.argmax(unassigned)]  # smallest position still unassigned
                dist = np.abs(S[run] - S[lead]).max(axis=1)
                match = unassigned & (dist <= tol_sig)
                if not unassigned.all() or not match.all():
                    far = dist[unassigned & ~match]
                    if far.size:
                        margins["min_between_sig"] = min(margins["min_between_sig"], float(far.min()))
                leader_of[run[match]] = lead
                margins["max_within_sig"] = max(margins["max_within_sig"], float(dist[match].max()))
                margins["max_within_F"] = max(margins["max_within_F"], float(np.abs(F[run[match]] - F[lead]).max()))
                unassigned &= ~match
                run_leaders.append(int(lead))
                leaders.append(int(lead))
            if g_canon is not None:
                G = np.asarray(g_canon)
                for lead in run_leaders:
                    dg = np.abs(G[run] - G[lead]).reshape(run.size, -1).max(axis=1)
                    same = leader_of[run] == lead
                    margins["max_within_g"] = max(margins["max_within_g"], float(dg[same].max()))
                    if (~same).any():
                        margins["min_between_g"] = min(margins["min_between_g"], float(dg[~same].min()))
                    assert ((dg <= tol_g) == same).all(), "signature partition and configuration partition differ"
    leaders = np.array(sorted(leaders), dtype=np.int64)
    copy_id[keep] = np.searchsorted(leaders, leader_of[keep])
    n_distinct = int(leaders.size)
    multiplicity = np.bincount(copy_id[keep], minlength=n_distinct).astype(np.int64) if n_distinct else np.zeros(0, np.int64)
    hist = None
    if nbins:
        hist = np.zeros(nbins, dtype=np.int64)
        b = np.clip(np.floor(F[leaders] * nbins).astype(np.int64), 0, nbins - 1)
        np.add.at(hist, b, multiplicity)
    return dict(copy_id=copy_id, n_distinct=n_distinct, rep=leaders, multiplicity=multiplicity, hist=hist,
                F_rep=F[leaders], margins=margins)


def discovery_curve(rep, n_levels):
    """SURVEY 8(f)-1, PAPER.md:L149 / Figs. 1-3: curve[k] = number of copies whose first discovery (leader position,
    `rep` as returned by count_copies) lies among the first 2^k samples, written out as the definition."""
    rep = [int(r) for r in np.asarray(rep).ravel()]
    return np.array([sum(1 for r in rep if r < (1 << k)) for k in range(int(n_levels))], dtype=np.int64)


def paper_count(F_norm, status, scale=1e8):
    """the paper converts x = 1 - F/(dV) into the integer X = floor(x * 1e8) and counts the
    distinct integers among its converged samples."""
    keys = set()
    for f, st in zip(np.asarray(F_norm, dtype=np.float64).ravel(), np.asarray(status, dtype=np.uint8).ravel()):
        if (int(st) & 1) == 0:
            keys.add(int(np.floor((1.0 - float(f)) * float(scale))))
    return len(keys)



# ------------------------------------------------------------------------------------------------
# Ensemble read-outs: what the paper tabulates / plots from many orbits.  Plain loops.
# Per orbit the inputs are the outputs of count_copies on that orbit: F_rep[c] (F/(dV) of the leader of
# copy c) and multiplicity[c].  The paper's value of a minimum is x = 1 - F/(dV) (Eq. 3).
# ------------------------------------------------------------------------------------------------
def _mean_std(values):
    """Average and standard deviation as printed in Tab. I / III ("avg +- std"; the paper gives no formula --
    reading R18: sample standard deviation, n-1 in the denominator, 0 for one value), NaN entries left out."""
    v = [float(x) for x in values if not np.isnan(x)]
    if not v:
        return float("nan"), float("nan")
    s = 0.0
    for x in v:
        s = s + x
    mean = s / len(v)
    q = 0.0
    for x in v:
        e = x - mean
        q = q + e * e
    return mean, (float(np.sqrt(q / (len(v) - 1))) if len(v) > 1 else 0.0)


def ensemble_stats(F_rep_per_orbit, n_in_region=None):
    """Tab. I: average and standard deviation over the orbits of the number of distinct minima;
    Tab. III (L213-220): of the value at the global minimum, x_g = the smallest x found on the orbit (L169) =
    1 - max_c F_rep[c]; and of the number of copies inside the first Gribov region (L9, L50) when given.
    Returns dict(best_x [n_orbits], n_distinct=(mean, std), best=(mean, std), n_in_region=(mean, std), used)."""
    best = []
    for F in F_rep_per_orbit:
        F = np.asarray(F, dtype=np.float64)
        best.append(1.0 - float(F.max()) if F.size else float("nan"))
    nd = [float(np.asarray(F).size) for F in F_rep_per_orbit]
    return dict(best_x=np.array(best), n_distinct=_mean_std(nd), best=_mean_std(best),
                n_in_region=_mean_std([float(v) for v in n_in_region]) if n_in_region is not None else (float("nan"),) * 2,
                used=sum(1 for b in best if not np.isnan(b)))


def relative_deviation_hist(F_rep_per_orbit, multiplicity_per_orbit, dev_max, nbins):
    """Fig. 8: "the distribution of the minima F_i relative to the global minimum F_g on that
    orbit: (F_i - F_g)/F_g.  Subsequently, the data has been averaged over all orbits."  In the paper's convention the
    F there are the values x.  Every converged sample counts (a copy found m times puts m entries: the bins of Fig. 5
    scale with the number of samples, L167 -- reading R19).  nbins equal bins on [0, dev_max), larger values in the
    last bin.  Orbits without samples or with x_g = 0 (trivial orbit: no relative deviation) are left out.
    Returns dict(counts [n_orbits, nbins], n_converged [n_orbits], avg [nbins], used)."""
    n_orb = len(F_rep_per_orbit)
    counts = np.zeros((n_orb, nbins), dtype=np.int64)
    nconv = np.zeros(n_orb, dtype=np.int64)
    width = float(dev_max) / float(nbins)
    for o in range(n_orb):
        F = np.asarray(F_rep_per_orbit[o], dtype=np.float64)
        m = np.asarray(multiplicity_per_orbit[o], dtype=np.int64)
        if F.size == 0:
            continue
        xg = 1.0 - float(F.max())
        if not xg > 0.0:
            continue
        for c in range(F.size):
            x = 1.0 - float(F[c])
            dev = (x - xg) / xg
            q = int(np.floor(dev / width))
            b = 0 if q < 0 else (nbins - 1 if q >= nbins else q)
            counts[o, b] += int(m[c])
            nconv[o] += int(m[c])
    avg = np.zeros(nbins)
    used = 0
    for b in range(nbins):
        s, used = 0.0, 0
        for o in range(n_orb):
            if nconv[o] == 0:
                continue
            s = s + float(counts[o, b]) / float(nconv[o])
            used += 1
        avg[b] = s / used if used else 0.0
    return dict(counts=counts, n_converged=nconv, avg=avg, used=used)


def hist_ratio(hist_small, hist_big):
    """Fig. 5: "We assign each minimum to a bin of resolution 1e-4 and plot the ratios of the
    entries of the bins from 256 vs. four mebisamples"; "only very high-lying bins of the four mebisample run are empty
    while the corresponding bins of the 256 mebisample run have entries".  ratio[b] = big/small (inf where only the
    larger run has entries, NaN where neither); n_only = (bins only the larger run fills, bins only the smaller)."""
    ratio, only_big, only_small = [], 0, 0
    for s, g in zip(np.asarray(hist_small).tolist(), np.asarray(hist_big).tolist()):
        ratio.append(g / s if s > 0 else (float("inf") if g > 0 else float("nan")))
        only_big += 1 if (s == 0 and g > 0) else 0
        only_small += 1 if (g == 0 and s > 0) else 0
    return dict(ratio=np.array(ratio), n_only=(only_big, only_small))
