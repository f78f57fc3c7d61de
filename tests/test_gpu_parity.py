"""GPU parity tests (-m gpu): the CUDA path, called through the C-ABI binding, against the CPU oracle on the same
seeded inputs.  Bars (north_star / DESIGN.md section 6): integer outputs (sweeps, status, copy_id, counts, rep,
multiplicity, histogram, region) bit-exact; F/(dV) within 1e-10 absolute; lambda_1 within 1e-8; canonical
configurations within 1e-7 per component (same trajectory, different rounding order)."""
import numpy as np
import pytest

from paper_1403_0555_b200 import synth

pytestmark = pytest.mark.gpu

TOL_F = 1e-10
TOL_LAM = 1e-8
TOL_G = 1e-7


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1403_0555_b200 import binding
    binding.lib()
    return binding


def _cpu(t):
    return t.cpu().numpy()


def _compare_relax(o, r, V, *, exact_sweeps=True):
    """o: oracle dict, r: GPU dict of numpy arrays.  Any sweep mismatch is reported with its start index (R14)."""
    bad = np.nonzero(o["sweeps"] != r["sweeps"])[0]
    if exact_sweeps:
        assert bad.size == 0, f"sweeps differ at starts {bad[:10]}: oracle {o['sweeps'][bad[:10]]} gpu {r['sweeps'][bad[:10]]}"
    assert (o["status"] == r["status"]).all()
    assert np.abs(o["F_norm"] - r["F_norm"]).max() < TOL_F
    assert np.abs(o["sig"] - r["sig"]).max() < TOL_G
    if o.get("g_canon") is not None and r.get("g_canon") is not None:
        assert np.abs(o["g_canon"] - r["g_canon"]).max() < TOL_G


def _gpu_relax(b, orbit, seed, n, **kw):
    out = b.relax_batch(orbit, seed, n, **kw)
    return {k: (_cpu(v) if v is not None and k != "workspace" else None) for k, v in out.items() if k != "workspace"}


LATTICES = [
    ((4, 4), 1, 512), ((8, 8), 2, 256), ((4, 4, 4), 3, 256), ((4, 4, 4, 4), 12, 96), ((2, 2, 2, 2), 12, 512),
    ((3, 3, 3, 3), 12, 128), ((3, 2), 40, 256), ((2, 2), 41, 256), ((5, 3, 2), 7, 128), ((6, 6, 6, 6), 12, 12),
    ((8, 8, 8, 8), 12, 4), ((7,), 77, 128), ((6, 4), 5, 128), ((4, 6, 2, 3), 9, 32), ((10, 10), 8, 64),
    ((8, 8, 8), 21, 70), ((6, 6), 22, 300), ((6, 6, 6), 23, 40),
]


@pytest.mark.parametrize("ext,seed,n", LATTICES)
@pytest.mark.parametrize("kernel", [0, 1, 2, 3])
def test_relax_matches_oracle(b, oracle, ext, seed, n, kernel):
    """a2-a6 on hot orbits: every lattice shape the kernels dispatch on (resident specialisations, streamed large even
    lattices, generic even, generic odd-extent level phases, extent-2 double bonds, d = 1): the automatic choice, the
    generic kernel, and the streamed kernel forced onto every all-even lattice (refill and ragged teams included:
    n is not a multiple of 32 for some of them)."""
    tma = ext in ((6,) * 4, (8,) * 4)
    if kernel == 3 and not tma:
        pytest.skip("the TMA-staged streamed kernel exists for 6^4 and 8^4")
    th = synth.uniform_links(ext, seed)
    orbit = b.Orbit(ext, th)
    orbit.set_kernel(kernel)
    if kernel == 3:
        assert orbit.kernel_name == "tma_stream_lane_per_start"
        n = 3 * n + 5    # several refills per lane and a ragged last batch
    if kernel == 1 and orbit.kernel_name != "generic_cta_per_start":
        pytest.fail("set_kernel(1) must select the generic kernel")
    odd = any(e % 2 for e in ext)
    if kernel == 2 and orbit.kernel_name != ("phased_lane_per_start" if odd else "stream_lane_per_start"):
        pytest.fail("set_kernel(2) must select the streamed (all-even) / phased (odd extent) lane-per-start kernel")
    if kernel == 0 and orbit.V >= 1024 and not odd:   # 6^4, 8^4: the TMA-staged streamed kernel
        assert orbit.kernel_name == ("tma_stream_lane_per_start" if ext in ((6,) * 4, (8,) * 4) else "stream_lane_per_start")
    if kernel == 0 and orbit.V >= 64 and odd:
        assert orbit.kernel_name == "phased_lane_per_start"
    V = orbit.V
    eps = 1e-12 if V > 256 else 1e-13
    o = oracle.relax(ext, th, seed, n, eps=eps, want_g=True)
    r = _gpu_relax(b, orbit, seed, n, eps=eps, want_g=True)
    _compare_relax(o, r, V)
    assert (o["status"] == 0).all()


def test_relax_gaussian_orbits_and_omega(b, oracle):
    """Configs 2 / 4 orbit shape (Gaussian noise + random gauge transform); omega = 1 (the paper's setting, L99)
    and omega = 1.95."""
    for ext, seed, sigma, n in [((8, 8), 2, 0.6, 256), ((4, 4, 4, 4), 11, 0.8, 64)]:
        th = synth.gaussian_gauged_links(ext, seed, sigma)
        orbit = b.Orbit(ext, th)
        for omega in (1.0, 1.7, 1.95):
            o = oracle.relax(ext, th, seed, n, omega=omega, want_g=True)
            for kernel in (0, 2):                       # the resident kernel and the streamed one forced onto it
                orbit.set_kernel(kernel)
                r = _gpu_relax(b, orbit, seed, n, omega=omega, want_g=True)
                _compare_relax(o, r, orbit.V)


def test_relax_options(b, oracle):
    """start_ids, first_start, 64-bit seeds and start indices, check_every, max_sweeps (status bit0), n = 0."""
    ext = (4, 4, 4)
    th = synth.uniform_links(ext, 3)
    orbit = b.Orbit(ext, th)
    for kernel in (0, 1, 2):                            # resident, generic, streamed
        orbit.set_kernel(kernel)
        ids = np.array([5, 3, 2 ** 40 + 7, 3, 2 ** 63 + 11, 0], dtype=np.uint64)
        seed = (9 << 32) | 1234567
        _compare_relax(oracle.relax(ext, th, seed, 0, start_ids=ids, want_g=True),
                       _gpu_relax(b, orbit, seed, 0, start_ids=ids, want_g=True), 64)
        _compare_relax(oracle.relax(ext, th, 3, 100, first_start=1000), _gpu_relax(b, orbit, 3, 100, first_start=1000), 64)
        for ce in (2, 5):
            _compare_relax(oracle.relax(ext, th, 3, 128, check_every=ce), _gpu_relax(b, orbit, 3, 128, check_every=ce), 64)
        o = oracle.relax(ext, th, 3, 64, max_sweeps=10)
        r = _gpu_relax(b, orbit, 3, 64, max_sweeps=10)
        assert (r["status"] & 1).all() and (r["sweeps"] == 10).all()
        _compare_relax(o, r, 64)
        o = oracle.relax(ext, th, 3, 64, max_sweeps=40)          # a mix of converged and not
        r = _gpu_relax(b, orbit, 3, 64, max_sweeps=40)
        _compare_relax(o, r, 64)
        assert b.relax_batch(orbit, 3, 0)["F_norm"].numel() == 0
        with pytest.raises(b.U1gfError):
            b.relax_batch(orbit, 3, 4, omega=2.0)
        with pytest.raises(b.U1gfError):
            b.relax_batch(orbit, 3, 4, eps=0.0)


def test_relax_is_deterministic_and_batch_independent(b):
    """A start's result is a pure function of (orbit, seed, index): identical bits whether it runs alone, in a big
    batch, through start_ids or twice (include/u1gf.h contract; the representative re-relaxation relies on it)."""
    import torch
    for ext, seed in [((4, 4, 4, 4), 12), ((8, 8), 2), ((4, 4), 1), ((3, 3, 3, 3), 12), ((8, 8, 8), 21)]:
        orbit = b.Orbit(ext, synth.uniform_links(ext, seed))
        big = b.relax_batch(orbit, seed, 3000, want_g=False)
        again = b.relax_batch(orbit, seed, 3000)
        assert torch.equal(big["F_norm"], again["F_norm"]) and torch.equal(big["sig"], again["sig"])
        ids = np.array([2999, 17, 1024, 0, 777], dtype=np.uint64)
        sub = b.relax_batch(orbit, seed, 0, start_ids=ids)
        idx = torch.as_tensor(ids.astype(np.int64), device="cuda")
        assert torch.equal(sub["F_norm"], big["F_norm"][idx]) and torch.equal(sub["sweeps"], big["sweeps"][idx])
        assert torch.equal(sub["sig"], big["sig"][idx])
        one = b.relax_batch(orbit, seed, 1, first_start=1024)
        assert torch.equal(one["F_norm"][0], big["F_norm"][1024])


def test_host_entry_points(b, oracle):
    ext = (4, 4)
    th = synth.uniform_links(ext, 1)
    orbit = b.Orbit(ext, th)
    o = oracle.relax(ext, th, 1, 300, want_g=True)
    r = b.relax_batch_host(orbit, 1, 300, want_g=True)
    _compare_relax(o, r, 16)
    c = b.count_copies_host(r["F_norm"], r["sig"], r["status"], nbins=100)
    oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"], nbins=100)
    assert c["n_distinct"] == oc["n_distinct"] and (c["copy_id"] == oc["copy_id"]).all()
    assert (c["hist"] == oc["hist"]).all()
    f = b.check_fp_host(orbit, r["g_canon"][c["rep"]])
    for k, rep in enumerate(c["rep"]):
        lam, region = oracle.fp_lambda1(ext, th, o["g_canon"][rep])
        assert abs(f["lambda1"][k] - lam) < TOL_LAM and f["region"][k] == region
    assert f["n_in_region"] == len(c["rep"])


# ------------------------------------------------------------------------------------------------- a8
def _gpu_count(b, F, sig, status, **kw):
    import torch
    dev = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt, device="cuda")
    c = b.count_copies(dev(F, torch.float64), dev(np.asarray(sig).reshape(-1, 4), torch.float64),
                       dev(status, torch.uint8), **kw)
    nd = int(c["n_distinct"].item())
    return dict(copy_id=_cpu(c["copy_id"]), n_distinct=nd, rep=_cpu(c["rep"])[:nd],
                multiplicity=_cpu(c["multiplicity"])[:nd], hist=None if c["hist"] is None else _cpu(c["hist"]))


def _same_count(g, o):
    assert g["n_distinct"] == o["n_distinct"]
    assert (g["copy_id"] == o["copy_id"]).all()
    assert (g["rep"] == o["rep"]).all() and (g["multiplicity"] == o["multiplicity"]).all()
    if o["hist"] is not None:
        assert (g["hist"] == o["hist"]).all()


def test_count_copies_hand_made_records(b, oracle):
    sA, sB, sC = np.array([.1, .2, .3, .4]), np.array([.1, .2, .3, .4]) + 0.01, np.array([-.3, .2, .1, 0])
    F = np.array([0.50, 0.70, 0.50 + 2e-11, 0.50, 0.70 + 5e-11, 0.9, 0.50 - 3e-11, 0.70])
    sig = np.array([sA, sC, sA + 1e-6, sB, sC - 2e-5, sA, sB + 1e-5, sA])
    status = np.array([0, 0, 0, 0, 0, 1, 0, 2], dtype=np.uint8)
    g = _gpu_count(b, F, sig, status, nbins=10)
    assert g["copy_id"].tolist() == [0, 1, 0, 2, 1, -1, 2, 3]
    assert g["rep"].tolist() == [0, 1, 3, 7] and g["multiplicity"].tolist() == [2, 2, 2, 1]
    assert g["hist"].tolist() == [0, 0, 0, 0, 0, 4, 0, 3, 0, 0]
    _same_count(g, oracle.count_copies(F, sig, status, nbins=10))
    F2 = np.array([0.3, 0.3 + 0.8e-10, 0.3 + 1.6e-10, 0.3 + 2.8e-10])          # chained run
    g2 = _gpu_count(b, F2, np.tile(sA, (4, 1)), np.zeros(4, np.uint8))
    assert g2["copy_id"].tolist() == [0, 0, 0, 1]
    g0 = _gpu_count(b, np.zeros(0), np.zeros((0, 4)), np.zeros(0, np.uint8), nbins=4)   # empty
    assert g0["n_distinct"] == 0 and g0["hist"].tolist() == [0, 0, 0, 0]
    g1 = _gpu_count(b, np.array([0.2, 0.4]), np.zeros((2, 4)), np.ones(2, np.uint8), nbins=4)   # nothing converged
    assert g1["n_distinct"] == 0 and g1["copy_id"].tolist() == [-1, -1] and g1["hist"].sum() == 0
    gn = _gpu_count(b, np.array([-0.25, 0.4, -0.25]), np.zeros((3, 4)), np.zeros(3, np.uint8), nbins=4)  # negative F
    assert gn["copy_id"].tolist() == [0, 1, 0] and gn["hist"].tolist() == [2, 1, 0, 0]


def test_count_copies_random_records_bit_exact(b, oracle):
    """Adversarial synthetic records: many copies with equal F and different signatures (several election rounds),
    near-tolerance gaps, unconverged records sprinkled in; several sizes spanning many CTAs and a ragged tail."""
    rng = np.random.default_rng(5)
    for n, n_levels, n_sigs in [(1, 1, 1), (33, 3, 2), (1000, 10, 4), (70001, 300, 5), (300007, 5, 40)]:
        levels = rng.uniform(0.1, 0.9, n_levels)
        sigs = rng.uniform(-0.5, 0.5, (n_sigs, 4))
        li, si = rng.integers(0, n_levels, n), rng.integers(0, n_sigs, n)
        F = levels[li] + rng.uniform(-2e-11, 2e-11, n)
        sig = sigs[si] + rng.uniform(-2e-5, 2e-5, (n, 4))
        status = (rng.uniform(size=n) < 0.05).astype(np.uint8) | (2 * (rng.uniform(size=n) < 0.1)).astype(np.uint8)
        _same_count(_gpu_count(b, F, sig, status, nbins=1000), oracle.count_copies(F, sig, status, nbins=1000))


def test_pipeline_copy_assignment_matches_oracle(b, oracle):
    """relax -> count on both sides from the same seeds: identical start -> copy assignment, distinct-copy counts,
    multiplicities, histogram; per-copy F/(dV) within 1e-10; lambda_1 of every copy within 1e-8, same region."""
    cases = [((4, 4), "uniform", 1, 4096, None), ((8, 8), "gauss", 2, 4096, 0.6), ((4, 4, 4), "uniform", 3, 4096, None),
             ((2, 2, 2, 2), "uniform", 12, 2048, None), ((3, 3, 3, 3), "uniform", 12, 1024, None),
             ((4, 4, 4, 4), "gauss", 11, 512, 0.8), ((4, 4, 4, 4), "uniform", 12, 512, None), ((5, 5), "cold", 9, 2048, None)]
    for ext, kind, seed, n, sigma in cases:
        th = synth.make_theta(dict(extents=ext, kind=kind, seed=seed, sigma=sigma))
        orbit = b.Orbit(ext, th)
        eps = 1e-12 if (kind == "uniform" and len(ext) == 4) else 1e-13
        o = oracle.relax(ext, th, seed, n, eps=eps, want_g=True)
        oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"], nbins=10000, g_canon=o["g_canon"])
        r = b.relax_batch(orbit, seed, n, eps=eps)
        c = b.count_copies(r["F_norm"], r["sig"], r["status"], nbins=10000)
        nd = int(c["n_distinct"].item())
        assert nd == oc["n_distinct"], (ext, nd, oc["n_distinct"])
        assert (_cpu(c["copy_id"]) == oc["copy_id"]).all()
        rep = _cpu(c["rep"])[:nd]
        assert (rep == oc["rep"]).all() and (_cpu(c["multiplicity"])[:nd] == oc["multiplicity"]).all()
        assert (_cpu(c["hist"]) == oc["hist"]).all()
        assert np.abs(_cpu(r["F_norm"])[rep] - oc["F_rep"]).max() < TOL_F
        # representatives re-relaxed with their fields, then the FP test
        rr = b.relax_batch(orbit, seed, 0, start_ids=rep.astype(np.uint64), eps=eps, want_g=True)
        assert (_cpu(rr["F_norm"]) == _cpu(r["F_norm"])[rep]).all()          # bit-identical re-run
        f = b.check_fp(orbit, rr["g_canon"])
        lam_gpu, reg_gpu = _cpu(f["lambda1"]), _cpu(f["region"])
        n_check = min(nd, 200)
        for k in range(n_check):
            lam, region = oracle.fp_lambda1(ext, th, o["g_canon"][rep[k]])
            assert abs(lam_gpu[k] - lam) < TOL_LAM, (ext, k, lam_gpu[k], lam)
            assert reg_gpu[k] == region
        assert int(f["n_in_region"].item()) == int((reg_gpu != 0).sum())


# ------------------------------------------------------------------------------------------------- a7
def test_check_fp_closed_forms_and_regions(b, oracle):
    """Cold-orbit twists (closed-form spectrum; regions 1, 2 and 0), random non-stationary fields, d = 1 ring."""
    import torch
    import anglemath as am
    cases = [((5, 5), (1, 0)), ((6, 6), (1, 0)), ((6, 6), (2, 0)), ((4, 4), (1, 0)), ((6, 6, 6), (1, 0, 1)),
             ((8, 8), (3, 1)), ((6, 6), (2, 2)), ((4, 4, 4, 4), (0, 0, 0, 0)), ((4, 4, 4, 4), (1, 0, 0, 0)),
             ((6, 6, 6, 6), (1, 0, 0, 1)), ((8, 8, 8, 8), (1, 0, 0, 0)), ((2, 2), (0, 0)), ((12,), (1,))]
    for ext, k in cases:
        V, d, N = int(np.prod(ext)), len(ext), ext[0]
        th = synth.cold_links(ext)
        x = am.coords(ext)
        phi = 2 * np.pi * sum(k[mu] * x[:, mu] / ext[mu] for mu in range(d))
        g = am.to_g(phi)
        orbit = b.Orbit(ext, th)
        f = b.check_fp(orbit, torch.as_tensor(g[None], device="cuda"))
        c = np.array([np.cos(2 * np.pi * km / N) for km in k])
        spec = [sum(2 * c[mu] * (1 - np.cos(2 * np.pi * m[mu] / N)) for mu in range(d))
                for m in np.ndindex(*ext) if any(m)]
        lam = float(f["lambda1"][0])
        assert abs(lam - min(spec)) < TOL_LAM, (ext, k, lam, min(spec))
        expect = 1 if min(spec) > 1e-8 else (2 if abs(min(spec)) <= 1e-8 else 0)
        assert int(f["region"][0]) == expect and int(f["n_in_region"].item()) == (expect != 0)
    for ext, seed in [((4, 4), 1), ((4, 4, 4), 3), ((3, 3, 3, 3), 12), ((4, 4, 4, 4), 12), ((3, 2), 4), ((8, 8), 2)]:
        V = int(np.prod(ext))
        th = synth.uniform_links(ext, seed)
        orbit = b.Orbit(ext, th)
        fields = np.stack([oracle.start(V, seed, 100 + k) for k in range(24)])
        f = b.check_fp(orbit, torch.as_tensor(fields, device="cuda"))
        for k in range(24):
            lam, region = oracle.fp_lambda1(ext, th, fields[k])
            assert abs(float(f["lambda1"][k]) - lam) < TOL_LAM and int(f["region"][k]) == region
    e = b.check_fp(b.Orbit((4, 4), synth.cold_links((4, 4))), torch.zeros((0, 16, 2), dtype=torch.float64, device="cuda"))
    assert e["lambda1"].numel() == 0 and int(e["n_in_region"].item()) == 0


# --------------------------------------------------------------------------------- full-size sampled parity
@pytest.mark.parametrize("cfg,orbit_idx,n_sample", [(2, 0, 1500), (3, 0, 1500), (4, 0, 400), (5, 2, 300), (5, 3, 24), (5, 4, 6)])
def test_full_size_configs_sampled(b, oracle, cfg, orbit_idx, n_sample):
    """BASELINE configs at their full start counts in the launch configuration bench.py times; the oracle
    recomputes a random sample of start indices one by one (a start is a pure function of its index)."""
    import torch
    conf = synth.CONFIGS[cfg]
    ob = conf["orbits"][orbit_idx]
    ext, seed, n = ob["extents"], ob["seed"], ob["n_starts"]
    th = synth.make_theta(ob)
    orbit = b.Orbit(ext, th)
    r = b.relax_batch(orbit, seed, n, omega=conf["omega"], eps=conf["eps"], max_sweeps=conf["max_sweeps"])
    c = b.count_copies(r["F_norm"], r["sig"], r["status"], nbins=10000)
    ids = np.unique(np.concatenate([[0, n - 1], np.random.default_rng(cfg).integers(0, n, n_sample)]))
    o = oracle.relax(ext, th, seed, 0, start_ids=ids.astype(np.uint64), omega=conf["omega"], eps=conf["eps"],
                     max_sweeps=conf["max_sweeps"])
    F, sw, st, sig = (_cpu(r[k])[ids] for k in ("F_norm", "sweeps", "status", "sig"))
    bad = np.nonzero(sw != o["sweeps"])[0]
    assert bad.size == 0, f"sweeps differ at starts {ids[bad][:10]}"
    assert (st == o["status"]).all() and np.abs(F - o["F_norm"]).max() < TOL_F and np.abs(sig - o["sig"]).max() < TOL_G
    # properties that hold at any size
    nd = int(c["n_distinct"].item())
    cid, mult, rep = _cpu(c["copy_id"]), _cpu(c["multiplicity"])[:nd], _cpu(c["rep"])[:nd]
    Fall, stall = _cpu(r["F_norm"]), _cpu(r["status"])
    assert mult.sum() == int(((stall & 1) == 0).sum()) and int(_cpu(c["hist"]).sum()) == mult.sum()
    assert (cid[rep] == np.arange(nd)).all() and (np.diff(rep) > 0).all()          # discovery order
    conv = cid >= 0
    assert np.abs(Fall[conv] - Fall[rep[cid[conv]]]).max() <= 1e-9                  # members share their leader's F
    assert (np.bincount(cid[conv], minlength=nd) == mult).all()
    # the sampled starts fall into the same copies as on the oracle side: same partition of the sample
    oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"])
    gpu_ids = cid[ids]
    pairs = set(zip(gpu_ids.tolist(), oc["copy_id"].tolist()))
    assert len(pairs) == len(set(gpu_ids.tolist())) == len(set(oc["copy_id"].tolist()))


@pytest.mark.gpu
def test_discovery_curve_and_paper_count_match_oracle(b, oracle):
    """SURVEY 8(f)-1 through the C-ABI: integer outputs, bit-exact against the oracle on the same device-produced
    F / rep arrays (hot 4^3: hundreds of copies; 4x4: few copies; an empty batch)."""
    import torch
    for ext, seed, n in (((4, 4, 4), 3, 20000), ((4, 4), 1, 4096)):
        orbit = b.Orbit(ext, synth.uniform_links(ext, seed))
        r = b.relax_batch(orbit, seed, n)
        c = b.count_copies(r["F_norm"], r["sig"], r["status"])
        nd = int(c["n_distinct"].item())
        rep = _cpu(c["rep"])[:nd]
        for levels in (1, 16, 65):
            cur = _cpu(b.discovery_curve(c["rep"], nd, levels))
            assert (cur == oracle.discovery_curve(rep, levels)).all()
        assert cur[-1] == nd
        F, st = _cpu(r["F_norm"]), _cpu(r["status"])
        for scale in (1e8, 1e4):
            assert int(b.paper_count(r["F_norm"], r["status"], scale).item()) == oracle.paper_count(F, st, scale)
        st2 = r["status"].clone()
        st2[::3] |= 1                                    # not-converged records are ignored
        assert int(b.paper_count(r["F_norm"], st2).item()) == oracle.paper_count(F, _cpu(st2))
    e = torch.zeros(0, dtype=torch.float64, device="cuda")
    assert int(b.paper_count(e, torch.zeros(0, dtype=torch.uint8, device="cuda")).item()) == 0
    assert _cpu(b.discovery_curve(torch.zeros(1, dtype=torch.int64, device="cuda"), 0, 4)).tolist() == [0, 0, 0, 0]
    with pytest.raises(b.U1gfError):
        b.discovery_curve(torch.zeros(1, dtype=torch.int64, device="cuda"), 1, 66)


@pytest.mark.gpu
def test_omega_changes_basins_not_copies_on_gpu(b):
    """SURVEY 8(f)-2 / pin P12 at GPU scale: omega = 1 (the paper's relaxation) and omega = 1.7 find the
    same copies on saturated small orbits (the set of F/(dV) values agrees to 1e-9) while the start -> copy map and
    the multiplicities differ (on these tiny lattices plain relaxation even needs fewer sweeps)."""
    import torch
    for ext, seed, n in (((4, 4), 1, 1 << 16), ((2, 2, 2, 2), 12, 1 << 16)):
        orbit = b.Orbit(ext, synth.uniform_links(ext, seed))
        tables = {}
        for omega in (1.0, 1.7):
            r = b.relax_batch(orbit, seed, n, omega=omega)
            c = b.count_copies(r["F_norm"], r["sig"], r["status"])
            nd = int(c["n_distinct"].item())
            F = np.sort(_cpu(r["F_norm"])[_cpu(c["rep"])[:nd]])
            tables[omega] = (F, _cpu(c["copy_id"]), float(r["sweeps"].float().mean().item()), np.sort(_cpu(c["multiplicity"])[:nd]))
            assert int((r["status"] & 1).sum().item()) == 0
        F1, id1, sw1, m1 = tables[1.0]
        F17, id17, sw17, m17 = tables[1.7]
        assert F1.size == F17.size and np.abs(F1 - F17).max() < 1e-9
        assert sw1 != sw17                                 # a different path to the same copies ...
        assert (m1 != m17).any()                           # ... into basins of different sizes (the bias of L99)


@pytest.mark.gpu
@pytest.mark.parametrize("ext,seed,n,kind", [
    ((4, 4, 4, 4), 12, 1 << 17, "uniform"), ((4, 4, 4, 4), 11, 1 << 17, "gauss0.8"), ((4, 4, 4), 3, 1 << 18, "uniform"),
    ((8, 8), 2, 1 << 18, "gauss0.6"), ((2, 2, 2, 2), 12, 1 << 18, "uniform"), ((4, 4), 1, 1 << 18, "uniform"),
    ((6, 6, 6, 6), 12, 1 << 12, "uniform"), ((3, 3, 3, 3), 12, 1 << 16, "uniform"), ((8, 8, 8, 8), 12, 1 << 9, "uniform")])
def test_large_batches_element_by_element(b, oracle, ext, seed, n, kind):
    """Every start of a large batch against the oracle (10^5 .. 3 10^5 starts on the resident kernels, thousands on the
    big lattices): identical sweeps and status, F/(dV) within 1e-10, and the same copy id for every start -- up to 6 10^4
    distinct copies on the hot 4^4 orbit.  This is where a rounding-level difference between the two arithmetic paths
    (FMA contraction, second-order rsqrt polish, tree gauge, summation order) would show up as a sweep or a copy (R14)."""
    th = synth.uniform_links(ext, seed) if kind == "uniform" else synth.gaussian_gauged_links(ext, seed, float(kind[5:]))
    orbit = b.Orbit(ext, th)
    eps = 1e-12 if orbit.V > 256 else 1e-13
    o = oracle.relax(ext, th, seed, n, eps=eps)
    r = b.relax_batch(orbit, seed, n, eps=eps)
    sw, F, st, sg = (_cpu(r[k]) for k in ("sweeps", "F_norm", "status", "sig"))
    bad = np.nonzero(sw != o["sweeps"])[0]
    assert bad.size == 0, f"sweeps differ at starts {bad[:10]}: oracle {o['sweeps'][bad[:10]]} gpu {sw[bad[:10]]}"
    assert (st == o["status"]).all()
    assert np.abs(F - o["F_norm"]).max() < TOL_F and np.abs(sg - o["sig"]).max() < TOL_G
    c = b.count_copies(r["F_norm"], r["sig"], r["status"])
    oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"])
    assert int(c["n_distinct"].item()) == oc["n_distinct"]
    assert (_cpu(c["copy_id"]) == oc["copy_id"]).all()


@pytest.mark.gpu
@pytest.mark.parametrize("ext,seed,n", [((4, 4, 4, 4), 12, 1200), ((4, 4, 4), 3, 4000), ((6, 6, 6, 6), 12, 24), ((3, 3, 3, 3), 12, 600)])
def test_check_fp_every_copy_of_a_batch(b, oracle, ext, seed, n):
    """a7 on every distinct copy of a hot batch (about 1000 copies at 4^4): lambda_1 of the batched Lanczos kernel against
    the oracle's dense eigenvalue within 1e-8 (observed: 1e-13), identical region flags."""
    th = synth.uniform_links(ext, seed)
    orbit = b.Orbit(ext, th)
    eps = 1e-12 if orbit.V > 256 else 1e-13
    r = b.relax_batch(orbit, seed, n, eps=eps, want_g=True)
    c = b.count_copies(r["F_norm"], r["sig"], r["status"])
    nd = int(c["n_distinct"].item())
    g = r["g_canon"][c["rep"][:nd]].contiguous()
    f = b.check_fp(orbit, g)
    lam, reg, gh = _cpu(f["lambda1"]), _cpu(f["region"]), _cpu(g)
    for k in range(nd):
        lo, ro = oracle.fp_lambda1(ext, th, gh[k])
        assert abs(lo - lam[k]) < 1e-8 and ro == reg[k], f"copy {k}: oracle {lo} gpu {lam[k]}"
    assert int(f["n_in_region"].item()) == int((reg != 0).sum())
