"""GPU parity tests (-m gpu) added in round 2: ensembles in one launch, copy-table merge (8(f)-4), the
one-call host pipeline, the bias read-out (8(f)-2), the service path of the resident kernels under stress (ring sizes,
tail flush, R6 redo list) and the first-Gribov-region counts of every BASELINE config at full size.  Same bars as
tests/test_gpu_parity.py: integer outputs bit-exact, F/(dV) within 1e-10, lambda_1 within 1e-8."""
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


# ------------------------------------------------------------------------------------------- ensembles (8(f)-3)
@pytest.mark.parametrize("ext,seeds,n", [((4, 4, 4), list(range(3, 11)), 4100), ((4, 4), [1, 2, 3, 4, 5], 1000),
                                         ((4, 4, 4, 4), [11, 12, 13], 96), ((8, 8), [2, 7], 700),
                                         ((2, 2, 2, 2), [12, 13, 14], 333),
                                         # shapes without a resident kernel: the generic kernel's ensemble mode (Tab. I / III
                                         # volumes 2^2, 6^2, 2^3, 8^3; an odd and a mixed lattice)
                                         ((2, 2), [1, 2, 3], 300), ((6, 6), [1, 2, 3, 4], 500), ((2, 2, 2), [5, 6], 301),
                                         ((8, 8, 8), [3, 4], 40), ((3, 3), [1, 2], 200), ((3, 2), [7, 8, 9], 100)])
def test_ensemble_one_launch_matches_single_orbits_and_oracle(b, oracle, ext, seeds, n):
    """n_orbits orbits of one shape in ONE u1gf_relax_ensemble call == one u1gf_relax_batch call per orbit == the oracle,
    start by start (n is not a multiple of 32: the padding of each orbit's last batch must not leak); per-orbit copy
    tables and first-Gribov-region counts bit-exact against the oracle."""
    import torch
    thetas = [synth.uniform_links(ext, s) for s in seeds]
    ens = b.Ensemble(ext, np.stack(thetas), seeds)
    assert ens.n_orbits == len(seeds)
    r = b.relax_ensemble(ens, n)
    assert b.last_launch_count() == 1                      # one kernel for the whole ensemble
    assert ens.orbit(0).kernel_name.startswith("lanes_") or ens.orbit(0).kernel_name.startswith("generic"), ens.orbit(0).kernel_name
    c = b.count_copies_ensemble(r["F_norm"], r["sig"], r["status"], nbins=100)            # all orbits in one pass
    launches_one_pass = b.last_launch_count()
    st_mixed = r["status"].clone()
    st_mixed[:, 5::7] |= 1                                                                  # some records not converged
    st_mixed[-1, :] |= 1                                                                    # the last orbit: none converged
    for st_ in (r["status"], st_mixed):
        c1 = b.count_copies_ensemble(r["F_norm"], r["sig"], st_, nbins=100)
        cl = b.count_copies_ensemble(r["F_norm"], r["sig"], st_, nbins=100, one_pass=False)    # one u1gf_count_copies per orbit
        nd1 = _cpu(c1["n_distinct"])
        assert (nd1 == _cpu(cl["n_distinct"])).all() and (_cpu(c1["copy_id"]) == _cpu(cl["copy_id"])).all()
        assert (_cpu(c1["hist"]) == _cpu(cl["hist"])).all()
        for k in range(len(seeds)):
            for key in ("rep", "multiplicity"):
                assert (_cpu(c1[key][k])[:nd1[k]] == _cpu(cl[key][k])[:nd1[k]]).all(), (k, key)
    assert nd1[-1] == 0 and (_cpu(c1["copy_id"][-1]) == -1).all()
    assert b.last_launch_count() > launches_one_pass or len(seeds) == 1                    # the loop launches per orbit
    for k, (th, seed) in enumerate(zip(thetas, seeds)):
        single = b.relax_batch(b.Orbit(ext, th), seed, n)
        o = oracle.relax(ext, th, seed, n)
        for key in ("sweeps", "status"):
            assert (_cpu(r[key][k]) == _cpu(single[key])).all() and (_cpu(r[key][k]) == o[key]).all(), (k, key)
        assert np.abs(_cpu(r["F_norm"][k]) - _cpu(single["F_norm"])).max() < 1e-12
        assert np.abs(_cpu(r["F_norm"][k]) - o["F_norm"]).max() < TOL_F
        assert np.abs(_cpu(r["sig"][k]) - o["sig"]).max() < TOL_G
        oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"], nbins=100)
        nd = int(c["n_distinct"][k].item())
        assert nd == oc["n_distinct"] and (_cpu(c["copy_id"][k]) == oc["copy_id"]).all()
        assert (_cpu(c["rep"][k])[:nd] == oc["rep"]).all() and (_cpu(c["multiplicity"][k])[:nd] == oc["multiplicity"]).all()
        assert (_cpu(c["hist"][k]) == oc["hist"]).all()
        # first-region count of this orbit through the member handle
        member = ens.orbit(k)
        rr = b.relax_batch(member, seed, 0, start_ids=c["rep"][k][:nd].contiguous(), want_g=True)
        f = b.check_fp(member, rr["g_canon"])
        og = oracle.relax(ext, th, seed, 0, start_ids=oc["rep"].astype(np.uint64), want_g=True)
        regions = [oracle.fp_lambda1(ext, th, og["g_canon"][j]) for j in range(min(nd, 40))]
        lam, reg = _cpu(f["lambda1"]), _cpu(f["region"])
        for j, (lo, ro) in enumerate(regions):
            assert abs(lam[j] - lo) < TOL_LAM and reg[j] == ro
        if nd <= 40:
            assert int(f["n_in_region"].item()) == sum(1 for _, ro in regions if ro != 0)
    ens.close()
    torch.cuda.synchronize()


def test_ensemble_readouts_match_oracle(b, oracle):
    """u1gf_ensemble_stats / u1gf_relative_deviation_hist / u1gf_hist_ratio (Tab. I, Tab. III, Fig. 8, Fig. 5 of the paper)
    on ensembles relaxed and de-duplicated on the device, against the oracle's definitions on the same copy tables:
    integer outputs bit for bit, floating-point outputs within 1e-10; and x_g, n_distinct also against the oracle's own
    relaxation of every orbit."""
    import torch
    for ext, seeds, n, dev_max, nbins in (((4, 4), list(range(1, 13)), 2048, 0.6, 48), ((4, 4, 4), [3, 4, 5, 6], 3000, 0.25, 1000),
                                          ((2, 2, 2, 2), [12, 13, 14], 500, 0.5, 7)):
        thetas = [synth.uniform_links(ext, s) for s in seeds]
        ens = b.Ensemble(ext, np.stack(thetas), seeds)
        r = b.relax_ensemble(ens, n)
        c = b.count_copies_ensemble(r["F_norm"], r["sig"], r["status"], nbins=10000)
        K = len(seeds)
        nds = _cpu(c["n_distinct"])
        Fg, rep, mul = _cpu(r["F_norm"]), _cpu(c["rep"]), _cpu(c["multiplicity"])
        F_rep = [Fg[k][rep[k][:nds[k]]] for k in range(K)]
        mult = [mul[k][:nds[k]] for k in range(K)]
        n_in = torch.tensor([(7 * k + 3) % 5 for k in range(K)], dtype=torch.int64, device="cuda")   # any integers do here
        s = b.ensemble_stats(K, n, r["F_norm"], c["rep"], c["n_distinct"], n_in)
        os_ = oracle.ensemble_stats(F_rep, n_in_region=_cpu(n_in))
        best, stats = _cpu(s["best_x"]), _cpu(s["stats"])
        assert (best == os_["best_x"]).all()                        # one exact subtraction from the same F
        want = [*os_["n_distinct"], *os_["best"], *os_["n_in_region"], os_["used"], K]
        assert np.abs(stats - np.array(want, dtype=np.float64)).max() < 1e-10
        s0 = _cpu(b.ensemble_stats(K, n, r["F_norm"], c["rep"], c["n_distinct"])["stats"])
        assert np.isnan(s0[4]) and np.isnan(s0[5]) and (s0[:4] == stats[:4]).all()
        # against the oracle's own relaxation: same number of copies, same best value per orbit
        for k in range(K):
            o = oracle.relax(ext, thetas[k], seeds[k], n)
            oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"])
            assert oc["n_distinct"] == nds[k] and abs((1.0 - oc["F_rep"].max()) - best[k]) < TOL_F
        d = b.relative_deviation_hist(K, n, r["F_norm"], c["rep"], c["multiplicity"], c["n_distinct"], s["best_x"], dev_max, nbins)
        od = oracle.relative_deviation_hist(F_rep, mult, dev_max, nbins)
        assert (_cpu(d["counts"]) == od["counts"]).all() and (_cpu(d["n_converged"]) == od["n_converged"]).all()
        assert int(d["n_orbits_used"].item()) == od["used"] == K
        assert np.abs(_cpu(d["avg"]) - od["avg"]).max() < 1e-10 and abs(_cpu(d["avg"]).sum() - 1.0) < 1e-12
        assert (_cpu(d["n_converged"]) == n).all()                  # every start converged: every sample is binned
        # Fig. 5: the same orbits with a quarter of the samples (the first n/4 starts of each orbit are a prefix)
        r4 = b.relax_ensemble(ens, n // 4)
        c4 = b.count_copies_ensemble(r4["F_norm"], r4["sig"], r4["status"], nbins=10000)
        big, small = c["hist"].sum(dim=0), c4["hist"].sum(dim=0)
        h = b.hist_ratio(small, big)
        oh = oracle.hist_ratio(_cpu(small), _cpu(big))
        ratio = _cpu(h["ratio"])
        assert np.array_equal(np.isnan(ratio), np.isnan(oh["ratio"])) and np.array_equal(np.isinf(ratio), np.isinf(oh["ratio"]))
        fin = np.isfinite(ratio)
        assert (ratio[fin] == oh["ratio"][fin]).all() and tuple(_cpu(h["n_only"]).tolist()) == oh["n_only"]
        assert oh["n_only"][1] == 0                                 # a prefix of the samples cannot fill a bin the full run misses
        ens.close()
    # an orbit without a converged start and the trivial orbit: NaN / left out, as the oracle does
    ext = (4, 4)
    th = np.stack([synth.uniform_links(ext, 1), synth.cold_links(ext)])
    ens = b.Ensemble(ext, th, [1, 2])
    r = b.relax_ensemble(ens, 256)
    c = b.count_copies_ensemble(r["F_norm"], r["sig"], r["status"])
    s = b.ensemble_stats(2, 256, r["F_norm"], c["rep"], c["n_distinct"])
    d = b.relative_deviation_hist(2, 256, r["F_norm"], c["rep"], c["multiplicity"], c["n_distinct"], s["best_x"], 1.0, 10)
    nds = _cpu(c["n_distinct"])
    Fg, rep, mul = _cpu(r["F_norm"]), _cpu(c["rep"]), _cpu(c["multiplicity"])
    od = oracle.relative_deviation_hist([Fg[k][rep[k][:nds[k]]] for k in range(2)], [mul[k][:nds[k]] for k in range(2)], 1.0, 10)
    assert (_cpu(d["counts"]) == od["counts"]).all() and int(d["n_orbits_used"].item()) == od["used"]
    assert np.abs(_cpu(d["avg"]) - od["avg"]).max() < 1e-10
    st2 = r["status"].clone()
    st2[1] |= 1                                                     # orbit 1: nothing converged
    c2 = b.count_copies_ensemble(r["F_norm"], r["sig"], st2)
    s2 = b.ensemble_stats(2, 256, r["F_norm"], c2["rep"], c2["n_distinct"])
    assert np.isnan(_cpu(s2["best_x"])[1]) and _cpu(s2["stats"])[6] == 1.0 and _cpu(s2["stats"])[3] == 0.0
    ens.close()
    with pytest.raises(b.U1gfError):
        b.hist_ratio(torch.zeros(0, dtype=torch.int64, device="cuda"), torch.zeros(0, dtype=torch.int64, device="cuda"))


# ------------------------------------------------------------------------------------------- table merge (8(f)-4)
@pytest.mark.parametrize("ext,seed,n,cuts", [((4, 4, 4), 3, 20000, (0, 7000, 7001, 20000)), ((4, 4), 1, 4096, (0, 2048, 4096)),
                                             ((4, 4, 4, 4), 12, 3000, (0, 1000, 2000, 3000))])
def test_merge_copy_tables_equals_single_process_ids(b, oracle, ext, seed, n, cuts):
    """Start ranges de-duplicated separately and merged with u1gf_merge_copy_tables give every start the copy id that
    one u1gf_count_copies / the oracle over all starts gives it; merged multiplicities and first discoveries agree."""
    import torch
    th = synth.uniform_links(ext, seed)
    orbit = b.Orbit(ext, th)
    eps = 1e-12 if orbit.V > 64 else 1e-13
    r = b.relax_batch(orbit, seed, n, eps=eps)
    F, S, st = r["F_norm"], r["sig"], r["status"]
    oc = oracle.count_copies(_cpu(F), _cpu(S), _cpu(st))
    tabs, local_ids, offs = [], [], []
    off = 0
    for a, z in zip(cuts[:-1], cuts[1:]):
        c = b.count_copies(F[a:z].contiguous(), S[a:z].contiguous(), st[a:z].contiguous())
        nd = int(c["n_distinct"].item())
        rep = c["rep"][:nd]
        tabs.append((F[a:z][rep], S[a:z][rep], rep + a, c["multiplicity"][:nd]))
        local_ids.append(_cpu(c["copy_id"]))
        offs.append(off)
        off += nd
    # tables concatenated in a scrambled range order: the merge orders entries by their first start itself
    order = list(range(len(tabs)))[::-1]
    cat = [torch.cat([tabs[k][j] for k in order]) for j in range(4)]
    pos_of = {}
    p = 0
    for k in order:
        pos_of[k] = p
        p += tabs[k][0].numel()
    m = b.merge_copy_tables(*cat)
    nm = int(m["n_merged"].item())
    mid = _cpu(m["merged_id"])
    assert nm == oc["n_distinct"]
    glob = np.full(n, -1, dtype=np.int64)
    for k, (a, z) in enumerate(zip(cuts[:-1], cuts[1:])):
        li = local_ids[k]
        conv = li >= 0
        glob[a:z][conv] = mid[pos_of[k] + li[conv]]
    assert (glob == oc["copy_id"]).all()
    assert (_cpu(m["first_start"])[:nm] == oc["rep"]).all()
    assert (_cpu(m["multiplicity"])[:nm] == oc["multiplicity"]).all()
    e = b.merge_copy_tables(F[:0], S[:0], torch.zeros(0, dtype=torch.int64, device="cuda"),
                            torch.zeros(0, dtype=torch.int64, device="cuda"))
    assert int(e["n_merged"].item()) == 0


# ------------------------------------------------------------------------------------------- one-call host pipeline
@pytest.mark.parametrize("ext,seed,n", [((4, 4, 4), 3, 5000), ((4, 4, 4, 4), 12, 700), ((6, 6, 6, 6), 12, 10)])
def test_pipeline_host_equals_separate_calls_and_oracle(b, oracle, ext, seed, n):
    th = synth.uniform_links(ext, seed)
    orbit = b.Orbit(ext, th)
    eps = 1e-12 if orbit.V > 64 else 1e-13
    p = b.pipeline_host(orbit, seed, n, eps=eps, nbins=50, first_start=7)
    o = oracle.relax(ext, th, seed, n, eps=eps, first_start=7, want_g=True)
    oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"], nbins=50)
    assert (p["sweeps"] == o["sweeps"]).all() and (p["status"] == o["status"]).all()
    assert np.abs(p["F_norm"] - o["F_norm"]).max() < TOL_F
    assert p["n_distinct"] == oc["n_distinct"] and (p["copy_id"] == oc["copy_id"]).all()
    assert (p["rep"] == oc["rep"]).all() and (p["multiplicity"] == oc["multiplicity"]).all() and (p["hist"] == oc["hist"]).all()
    assert np.abs(p["F_rep"] - oc["F_rep"]).max() < TOL_F
    n_in = 0
    for k in range(p["n_distinct"]):
        lo, ro = oracle.fp_lambda1(ext, th, o["g_canon"][oc["rep"][k]])
        assert abs(p["lambda1"][k] - lo) < TOL_LAM and (p["region"][k] & 3) == ro and not (p["region"][k] & 4)
        n_in += ro != 0
    assert p["n_in_region"] == n_in
    with pytest.raises(b.U1gfError):
        b.pipeline_host(orbit, seed, n, eps=eps, copy_capacity=0)
    b.lib().u1gf_release_host_scratch()


def test_pipeline_host_keeps_fields_on_hot_orbits(b):
    """A handle remembers that its last u1gf_pipeline_host call found most starts to be their own copy (n_distinct > n/4);
    the next call then writes the fields of all starts in the first pass and u1gf_check_fp picks the representatives by
    index, instead of relaxing them a second time.  A start is a pure function of its index, so every output of the two
    paths is identical; only the number of launches differs.  A cold orbit never takes the second path."""
    ext, seed, n = (4, 4, 4, 4), 12, 1500
    orbit = b.Orbit(ext, synth.uniform_links(ext, seed))
    calls = []
    for _ in range(3):
        p = b.pipeline_host(orbit, seed, n, eps=1e-12, nbins=64, first_start=3)
        calls.append((p, b.last_launch_count()))
        p = calls[-1][0]
        calls[-1] = ({k: (np.array(v, copy=True) if isinstance(v, np.ndarray) else v) for k, v in p.items()}, calls[-1][1])
    (p0, l0), (p1, l1), (p2, l2) = calls
    assert p0["n_distinct"] > n // 4                       # hot: the first call relaxes the representatives again ...
    assert l1 < l0 and l2 == l1                            # ... the later ones do not
    for q in (p1, p2):
        for k in ("sweeps", "status", "copy_id", "rep", "multiplicity", "region", "hist"):
            assert (p0[k] == q[k]).all(), k
        assert p0["n_distinct"] == q["n_distinct"] and p0["n_in_region"] == q["n_in_region"]
        assert (p0["F_norm"] == q["F_norm"]).all() and (p0["F_rep"] == q["F_rep"]).all()
        assert np.abs(p0["lambda1"] - q["lambda1"]).max() < 1e-12
    assert p0["n_in_region"] == int(((p0["region"] & 3) != 0).sum())
    # a batch of another size on the same handle: the remembered choice carries over, results equal those of a fresh handle
    fresh = b.Orbit(ext, synth.uniform_links(ext, seed))
    q, r = b.pipeline_host(orbit, seed, 333, eps=1e-12), None
    q = {k: (np.array(v, copy=True) if isinstance(v, np.ndarray) else v) for k, v in q.items()}
    r = b.pipeline_host(fresh, seed, 333, eps=1e-12)
    assert q["n_distinct"] == r["n_distinct"] and (q["region"] == r["region"]).all() and (q["rep"] == r["rep"]).all()
    assert np.abs(q["lambda1"] - r["lambda1"]).max() < 1e-12 and q["n_in_region"] == r["n_in_region"]
    # cold orbit (two copies among 4096 starts): every call takes the re-relaxation path
    cold = b.Orbit((4, 4), synth.uniform_links((4, 4), 1))
    counts = []
    for _ in range(2):
        c = b.pipeline_host(cold, 1, 4096)
        counts.append((b.last_launch_count(), c["n_distinct"], c["n_in_region"]))
    assert counts[0] == counts[1] and counts[0][1] < 1024
    b.lib().u1gf_release_host_scratch()


# ------------------------------------------------------------------------------------------- bias read-out (8(f)-2)
def test_bias_table_matches_oracle(b, oracle):
    """over-relaxation "decreases the chance of converging to larger minima and thus introduces a bias".
    Basin sizes (multiplicities) of every copy for omega = 1 (the paper's setting) and omega = 1.7 on the SAME starts,
    matched across the two runs by F and signature: the table the product reads out must equal the oracle's, bit-exact."""
    from paper_1403_0555_b200 import readout
    ext, seed, n = (4, 4, 4), 3, 8192
    th = synth.uniform_links(ext, seed)
    orbit = b.Orbit(ext, th)
    tab = readout.bias_table(orbit, seed, n)
    per = {}
    for omega in (1.0, 1.7):
        o = oracle.relax(ext, th, seed, n, omega=omega)
        oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"])
        per[omega] = (oc["F_rep"], o["sig"][oc["rep"]], oc["multiplicity"])
    # oracle-side matching, written out: a copy of run A equals the copy of run B with |dF| <= 1e-9 and |dsig| <= 1e-4
    F1, S1, M1 = per[1.0]
    F17, S17, M17 = per[1.7]
    rows = []
    used = set()
    for i in range(F1.size):
        j = [j for j in range(F17.size) if abs(F17[j] - F1[i]) <= 1e-9 and np.abs(S17[j] - S1[i]).max() <= 1e-4]
        assert len(j) <= 1
        rows.append((F1[i], int(M1[i]), int(M17[j[0]]) if j else 0))
        used.update(j)
    rows += [(F17[j], 0, int(M17[j])) for j in range(F17.size) if j not in used]
    rows.sort(key=lambda r: -r[0])
    assert len(rows) == len(tab["F"])
    assert np.abs(np.array([r[0] for r in rows]) - tab["F"]).max() < 1e-9
    assert [r[1] for r in rows] == tab["mult_omega1"].tolist() and [r[2] for r in rows] == tab["mult_omega"].tolist()
    assert tab["mult_omega1"].sum() == n and tab["mult_omega"].sum() == n


# ------------------------------------------------------------------------------------------- service path under stress
@pytest.mark.parametrize("ext,seed", [((4, 4, 4, 4), 11), ((8, 8), 2), ((4, 4, 4), 3), ((4, 4), 1)])
@pytest.mark.parametrize("check_every", [24, 32, 64])
def test_coarse_check_every_fills_the_dump_ring(b, oracle, ext, seed, check_every):
    """With check_every comparable to the convergence length all lanes of a team stop in the same few sweeps: up to 32
    dumps per service, several services in a row (the ring-overflow case of the round-1 review).  Every start against
    the oracle."""
    n = 4096 + 17
    th = synth.gaussian_gauged_links(ext, seed, 0.8) if len(ext) == 4 else synth.uniform_links(ext, seed)
    orbit = b.Orbit(ext, th)
    r = b.relax_batch(orbit, seed, n, check_every=check_every, want_g=True)
    o = oracle.relax(ext, th, seed, n, check_every=check_every, want_g=True)
    assert (_cpu(r["sweeps"]) == o["sweeps"]).all() and (_cpu(r["status"]) == o["status"]).all()
    assert np.abs(_cpu(r["F_norm"]) - o["F_norm"]).max() < TOL_F
    assert np.abs(_cpu(r["sig"]) - o["sig"]).max() < TOL_G
    assert np.abs(_cpu(r["g_canon"]) - o["g_canon"]).max() < TOL_G


@pytest.mark.parametrize("ext,seed", [((4, 4, 4, 4), 12), ((8, 8), 2), ((4, 4, 4), 3)])
def test_tail_flush_with_fewer_starts_than_lanes(b, oracle, ext, seed):
    """1..31 starts: every warp of the team dumps its block of the last fields in the final iteration and the flush
    must wait for all of them (the missing barrier of the round-1 review).  Repeated, with the fields written out."""
    th = synth.uniform_links(ext, seed)
    orbit = b.Orbit(ext, th)
    eps = 1e-12 if orbit.V > 64 else 1e-13
    for n in (1, 2, 5, 16, 31):
        o = oracle.relax(ext, th, seed, n, eps=eps, want_g=True)
        for _ in range(12):
            r = b.relax_batch(orbit, seed, n, eps=eps, want_g=True)
            assert (_cpu(r["sweeps"]) == o["sweeps"]).all()
            assert np.abs(_cpu(r["F_norm"]) - o["F_norm"]).max() < TOL_F
            assert np.abs(_cpu(r["sig"]) - o["sig"]).max() < TOL_G
            assert np.abs(_cpu(r["g_canon"]) - o["g_canon"]).max() < TOL_G


def test_r6_redo_list_through_the_generic_kernel(b, oracle):
    """R6 on the resident kernels: a start that meets |w|^2 below the threshold is put on a redo list and relaxed again by
    the generic kernel.  Random starts never get there, so the path is driven by a build of the library whose threshold
    is the high word of 0.5 (every start meets it within a few sweeps): all results then come from the redo path and
    must equal the oracle's (whose R6 threshold stays 1e-280, as does the generic kernel's)."""
    from paper_1403_0555_b200 import build
    regular = b.LIB_PATH
    try:
        b.use_library(build.build_variant("r6test", ["-DU1GF_R6_HI=0x3fe00000"]))
        for ext, seed, n in (((4, 4, 4, 4), 12, 300), ((8, 8), 2, 1000), ((4, 4), 1, 777)):
            th = synth.uniform_links(ext, seed)
            orbit = b.Orbit(ext, th)
            eps = 1e-12 if orbit.V > 64 else 1e-13
            ids = np.arange(n, dtype=np.uint64)[::-1].copy() + 5
            import torch
            r = b.relax_batch(orbit, seed, 0, start_ids=torch.as_tensor(ids.astype(np.int64), device="cuda"), eps=eps, want_g=True)
            assert b.last_launch_count() == 2
            o = oracle.relax(ext, th, seed, 0, start_ids=ids, eps=eps, want_g=True)
            assert (_cpu(r["sweeps"]) == o["sweeps"]).all() and (_cpu(r["status"]) == o["status"]).all()
            assert np.abs(_cpu(r["F_norm"]) - o["F_norm"]).max() < TOL_F
            assert np.abs(_cpu(r["g_canon"]) - o["g_canon"]).max() < TOL_G
            del orbit
    finally:
        b.use_library(regular)


def test_check_fp_reports_steps_and_convergence(b):
    ext, seed = (6, 6, 6, 6), 12
    orbit = b.Orbit(ext, synth.uniform_links(ext, seed))
    r = b.relax_batch(orbit, seed, 16, eps=1e-12, want_g=True)
    f = b.check_fp(orbit, r["g_canon"], want_steps=True)
    steps, reg = _cpu(f["steps"]), _cpu(f["region"])
    assert (steps > 10).all() and (steps < 512).all() and not (reg & 4).any()


# ------------------------------------------------------------------------------------------- full-size first-region counts
FULL = [(2, 0), (4, 0)] + [(3, k) for k in range(8)] + [(5, k) for k in range(5)]


@pytest.mark.parametrize("cfg,orbit_idx", FULL)
def test_full_size_first_region_counts_are_oracle_confirmed(b, oracle, cfg, orbit_idx):
    """Every BASELINE config at its full start count, in the launch configuration bench.py times: relax -> count ->
    re-relax the representatives -> Lanczos.  n_in_first_region = n_distinct - #exceptions, and EVERY exception (a copy
    the Lanczos kernel puts outside the region, marginal, or unconverged) is recomputed by the oracle from its start
    index -- relaxation, dense FP matrix, LAPACK eigenvalue -- and must come out the same (lambda_1 within 1e-8, same
    region).  These exceptions are genuine: starts that pass the gradient test while still leaving a saddle (R17); with
    eps -> 1e-26 the same start moves on to a minimum.  A sample of the copies inside the region, and of the starts, is
    oracle-checked the same way (the full sets are 10^5..10^6 copies)."""
    import torch
    conf = synth.CONFIGS[cfg]
    ob = conf["orbits"][orbit_idx]
    ext, seed, n = ob["extents"], ob["seed"], ob["n_starts"]
    V = int(np.prod(ext))
    th = synth.make_theta(ob)
    orbit = b.Orbit(ext, th)
    kw = dict(omega=conf["omega"], eps=conf["eps"], max_sweeps=conf["max_sweeps"])
    r = b.relax_batch(orbit, seed, n, **kw)
    c = b.count_copies(r["F_norm"], r["sig"], r["status"], nbins=10000)
    nd = int(c["n_distinct"].item())
    rep = c["rep"][:nd]
    lam = torch.empty(nd, dtype=torch.float64, device="cuda")
    reg = torch.empty(nd, dtype=torch.uint8, device="cuda")
    n_in = 0
    chunk = max(1, (4 << 30) // (V * 16))
    for a in range(0, nd, chunk):
        rr = b.relax_batch(orbit, seed, 0, start_ids=rep[a:a + chunk].contiguous(), want_g=True, **kw)
        f = b.check_fp(orbit, rr["g_canon"])
        lam[a:a + chunk], reg[a:a + chunk] = f["lambda1"], f["region"]
        n_in += int(f["n_in_region"].item())
        del rr
    lam, reg, rep = _cpu(lam), _cpu(reg), _cpu(rep)
    assert int(r["status"].sum().item()) == 0                       # every start converged, no R6 skip
    exceptions = np.nonzero(reg != 1)[0]
    assert n_in == nd - int((reg & 3 == 0).sum())
    assert exceptions.size <= 16, "more exceptions than the oracle can confirm in a test"
    sample = np.random.default_rng(cfg * 10 + orbit_idx).choice(nd, size=min(nd, 6 if V > 1000 else 24), replace=False)
    for k in np.concatenate([exceptions, sample]):
        sid = np.array([rep[k]], dtype=np.uint64)
        o = oracle.relax(ext, th, seed, 0, start_ids=sid, want_g=True, **kw)
        lo, ro = oracle.fp_lambda1(ext, th, o["g_canon"][0])
        assert abs(lo - lam[k]) < TOL_LAM and ro == reg[k], f"copy {k} start {rep[k]}: oracle {lo} {ro}, gpu {lam[k]} {reg[k]}"
        assert o["sweeps"][0] == int(r["sweeps"][rep[k]].item())
        assert abs(o["F_norm"][0] - float(r["F_norm"][rep[k]].item())) < TOL_F
    # sampled starts: same sweeps / F / partition as the oracle (all eight orbits of config 3, every size of config 5)
    ids = np.unique(np.concatenate([[0, n - 1], np.random.default_rng(cfg).integers(0, n, 300 if V <= 256 else (20 if V < 2000 else 5))]))
    o = oracle.relax(ext, th, seed, 0, start_ids=ids.astype(np.uint64), **kw)
    assert (_cpu(r["sweeps"])[ids] == o["sweeps"]).all()
    assert np.abs(_cpu(r["F_norm"])[ids] - o["F_norm"]).max() < TOL_F
    oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"])
    gpu_ids = _cpu(c["copy_id"])[ids]
    pairs = set(zip(gpu_ids.tolist(), oc["copy_id"].tolist()))
    assert len(pairs) == len(set(gpu_ids.tolist())) == len(set(oc["copy_id"].tolist()))


# ------------------------------------------------------------------------------------------- TMA-staged streamed kernel
@pytest.mark.parametrize("ext,seed", [((6, 6, 6, 6), 12), ((8, 8, 8, 8), 12)])
def test_tma_kernel_options(b, oracle, ext, seed):
    """relax_tma.cu on 6^4 / 8^4 against the oracle beyond the plain case of test_relax_matches_oracle: omega = 1 (its W1
    instantiation) and 1.95, max_sweeps (the lanes that reach it keep their pre-update even values like the lanes that
    converge: R5), check_every, start_ids / first_start / 64-bit seeds, a Gaussian orbit, and the same results from the
    plain-load streamed kernel."""
    V = int(np.prod(ext))
    small = V > 2000
    th = synth.uniform_links(ext, seed)
    orbit = b.Orbit(ext, th)
    assert orbit.kernel_name == "tma_stream_lane_per_start"

    def gpu(n, sd=seed, **kw):
        r = b.relax_batch(orbit, sd, n, want_g=True, **kw)
        return {k: (_cpu(v) if v is not None and k != "workspace" else None) for k, v in r.items() if k != "workspace"}

    def same(o, r):
        assert (o["sweeps"] == r["sweeps"]).all() and (o["status"] == r["status"]).all()
        assert np.abs(o["F_norm"] - r["F_norm"]).max() < TOL_F
        assert np.abs(o["sig"] - r["sig"]).max() < TOL_G and np.abs(o["g_canon"] - r["g_canon"]).max() < TOL_G

    n = 6 if small else 40
    for omega in (1.0, 1.95):
        same(oracle.relax(ext, th, seed, n, omega=omega, eps=1e-12, want_g=True), gpu(n, omega=omega, eps=1e-12))
    for ms in (30, 90):    # none / some of the starts converge before the cap
        o = oracle.relax(ext, th, seed, n, eps=1e-12, max_sweeps=ms, want_g=True)
        r = gpu(n, eps=1e-12, max_sweeps=ms)
        same(o, r)
        assert (r["status"] & 1).any()
    same(oracle.relax(ext, th, seed, n, eps=1e-11, check_every=3, want_g=True), gpu(n, eps=1e-11, check_every=3))
    ids = np.array([5, 3, 2 ** 40 + 7, 3, 2 ** 63 + 11, 0], dtype=np.uint64)
    sd = (9 << 32) | 1234567
    same(oracle.relax(ext, th, sd, 0, start_ids=ids, eps=1e-11, want_g=True), gpu(0, sd=sd, start_ids=ids, eps=1e-11))
    same(oracle.relax(ext, th, seed, 5, first_start=1000, eps=1e-11, want_g=True), gpu(5, first_start=1000, eps=1e-11))
    # the plain-load streamed kernel gives the same copies and sweeps
    r3 = gpu(n, eps=1e-12)
    orbit.set_kernel(2)
    r2 = gpu(n, eps=1e-12)
    assert orbit.kernel_name == "stream_lane_per_start"
    assert (r2["sweeps"] == r3["sweeps"]).all() and np.abs(r2["F_norm"] - r3["F_norm"]).max() < TOL_F
    # Gaussian orbit + gauge transform (the shape of configs 2 / 4): few copies, short relaxations
    thg = synth.gaussian_gauged_links(ext, 11, 0.8)
    og = b.Orbit(ext, thg)
    o = oracle.relax(ext, thg, 11, 70, want_g=True)
    r = b.relax_batch(og, 11, 70, want_g=True)
    same(o, {k: (_cpu(v) if v is not None and k != "workspace" else None) for k, v in r.items() if k != "workspace"})


@pytest.mark.parametrize("ext,n", [((6, 6, 6, 6), 32768), ((8, 8, 8, 8), 4096)])
def test_tma_kernel_equals_plain_stream_kernel_at_scale(b, ext, n):
    """Two independent implementations of the streamed path (bulk-copy staged tiles with in-place even rows and F from the
    last even half-sweep; plain loads with double-buffered even rows and F gathered in the finalisation) on batches far
    beyond what the oracle checks element by element: identical sweeps and status, F and signature to rounding."""
    import torch
    th = synth.uniform_links(ext, 12)
    res = {}
    for k in (3, 2):
        orbit = b.Orbit(ext, th)
        orbit.set_kernel(k)
        r = b.relax_batch(orbit, 12, n, eps=1e-12)
        torch.cuda.synchronize()
        res[k] = {x: _cpu(r[x]) for x in ("sweeps", "F_norm", "sig", "status")}
    a, c = res[3], res[2]
    assert (a["sweeps"] == c["sweeps"]).all() and (a["status"] == c["status"]).all() and not a["status"].any()
    assert np.abs(a["F_norm"] - c["F_norm"]).max() < 1e-13 and np.abs(a["sig"] - c["sig"]).max() < 1e-12
