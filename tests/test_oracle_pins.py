"""Pins for the CPU oracle (-m "not gpu"): each test checks the oracle against something the paper or the
mathematics fixes -- never against the oracle's own formulas.  P<k> numbers follow DESIGN.md section 4."""
import os

import numpy as np
import pytest
import scipy.linalg

import anglemath as am
from paper_1403_0555_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def hot(ext, seed):
    return synth.uniform_links(ext, seed)


def rand_phi(V, seed):
    return np.random.default_rng(seed).uniform(-np.pi, np.pi, V)


# ----------------------------------------------------------------------------------------------- P10
def test_philox_known_answers(oracle):
    """Philox4x32-10 (ref [59]) against the published known-answer vectors, and the oracle's
    C++ generator against the independent numpy one in synth.py."""
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        out = oracle.philox4x32_10(w[0:4], w[4:6])
        assert [int(v) for v in out] == w[6:10]
        out2 = synth.philox4x32_10(np.array([w[0]]), w[1], w[2], w[3], w[4], w[5])
        assert [int(v[0]) for v in out2] == w[6:10]


def test_start_is_uniform_philox_angle(oracle):
    """O2: g_i = exp(i pi (2u-1)), u the 53-bit uniform of Philox key (seed), counter (i, s_lo, s_hi, 0)."""
    V, seed, s = 81, (7 << 32) | 12345, (3 << 32) | 99
    g = oracle.start(V, seed, s)
    w = synth.philox4x32_10(np.arange(V, dtype=np.uint64), s & 0xFFFFFFFF, s >> 32, 0, seed & 0xFFFFFFFF, seed >> 32)
    u = (((w[1] << np.uint64(32)) | w[0]) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
    phi = np.pi * (2 * u - 1)
    assert np.abs(g[:, 0] - np.cos(phi)).max() < 1e-15 and np.abs(g[:, 1] - np.sin(phi)).max() < 1e-15
    assert np.abs(np.hypot(g[:, 0], g[:, 1]) - 1).max() < 4e-16
    # uniformity / independence smoke test over many starts
    ang = np.concatenate([am.to_phi(oracle.start(64, 5, k)) for k in range(400)])
    h, _ = np.histogram(ang, bins=16, range=(-np.pi, np.pi))
    assert abs(h - len(ang) / 16).max() < 5 * np.sqrt(len(ang) / 16)
    assert abs(np.corrcoef(ang[:-1], ang[1:])[0, 1]) < 0.03
    assert not np.allclose(oracle.start(16, 5, 0), oracle.start(16, 5, 1))
    assert not np.allclose(oracle.start(16, 5, 0), oracle.start(16, 6, 0))


# ------------------------------------------------------------------------------------------------ P1
@pytest.mark.parametrize("ext", [(2, 2), (3, 2), (4, 4), (5, 3, 2), (4, 4, 4), (3, 3, 3, 3), (2, 2, 2, 2), (4, 6, 2, 3), (7,)])
def test_angle_form_cross_check(oracle, ext):
    """Complex-arithmetic F, Delta_i and FP matrix equal the trigonometric angle forms (Eq. 3; L38)."""
    V = int(np.prod(ext))
    th = hot(ext, 21)
    phi = rand_phi(V, 22)
    F, vt, D = oracle.measure(ext, th, am.to_g(phi))
    assert abs(F - am.functional(ext, th, phi)) < 1e-12 * V
    Da = am.divergence(ext, th, phi)
    assert np.abs(D - Da).max() < 1e-13
    assert abs(vt - (Da ** 2).mean()) < 1e-13
    assert np.abs(oracle.fp_matrix(ext, th, am.to_g(phi)) - am.fp_matrix(ext, th, phi)).max() < 1e-13
    # links are (cos, sin) of the angles
    U = oracle.links(ext, th)
    assert np.abs(U[..., 0].reshape(-1) - np.cos(th)).max() == 0 and np.abs(U[..., 1].reshape(-1) - np.sin(th)).max() == 0


def test_gradient_and_hessian_by_finite_differences(oracle):
    """Delta = -dF/dphi and M = -d2F/dphi2 (f_i = dF/dg_i, M_FP = Hessian), central differences of
    the oracle's own F -- pins signs and the double-bond / odd-extent bookkeeping."""
    for ext in [(2, 2), (3, 2), (4, 3, 2)]:
        V = int(np.prod(ext))
        th = hot(ext, 31)
        phi = rand_phi(V, 32)
        Ff = lambda p: oracle.measure(ext, th, am.to_g(p))[0]
        _, _, D = oracle.measure(ext, th, am.to_g(phi))
        M = oracle.fp_matrix(ext, th, am.to_g(phi))
        e = 1e-5
        for i in range(V):
            ei = np.zeros(V); ei[i] = e
            assert abs((Ff(phi + ei) - Ff(phi - ei)) / (2 * e) + D[i]) < 1e-8
            for j in range(i, V):
                ej = np.zeros(V); ej[j] = e
                h = (Ff(phi + ei + ej) - Ff(phi + ei - ej) - Ff(phi - ei + ej) + Ff(phi - ei - ej)) / (4 * e * e)
                assert abs(h + M[i, j]) < 2e-5


# ------------------------------------------------------------------------------------------------ P2
def _polish(ext, th, phi, iters=60):
    """Newton on the angle form with phi_{V-1} pinned; returns (phi, converged, is_maximum)."""
    V = len(phi)
    phi = phi.copy()
    for _ in range(iters):
        D = am.divergence(ext, th, phi)[:-1]
        M = am.fp_matrix(ext, th, phi)[:-1, :-1]
        try:
            step = np.linalg.solve(M, D)
        except np.linalg.LinAlgError:
            return phi, False, False
        phi[:-1] -= step
        if np.abs(step).max() < 1e-14:
            break
    D = am.divergence(ext, th, phi)
    ok = np.abs(D).max() < 1e-11
    ev = np.linalg.eigvalsh(am.fp_matrix(ext, th, phi)[:-1, :-1])
    return phi, ok, bool(ok and ev[0] > 1e-9)


def _brute_force_maxima(ext, th, n_grid):
    """All local maxima of F over the V-1 free angles: dense grid scan -> grid-local maxima -> Newton polish ->
    keep maxima (grounded Hessian of -F positive definite) -> de-duplicate."""
    V = int(np.prod(ext))
    d = len(ext)
    grid = -np.pi + 2 * np.pi * np.arange(n_grid) / n_grid
    mesh = np.meshgrid(*([grid] * (V - 1)), indexing="ij")
    phis = list(mesh) + [np.zeros_like(mesh[0])]           # phi_{V-1} = 0
    idx = np.arange(V).reshape(am.shape(ext))
    tha = th.reshape(V, d)
    F = np.zeros(mesh[0].shape)
    for mu in range(d):
        j = np.roll(idx, -1, axis=am.axis(ext, mu)).reshape(-1)
        for i in range(V):
            F += np.cos(tha[i, mu] + phis[i] - phis[j[i]])
    is_max = np.ones(F.shape, dtype=bool)
    for ax in range(V - 1):
        is_max &= (F >= np.roll(F, 1, axis=ax)) & (F >= np.roll(F, -1, axis=ax))
    found = []
    for pt in np.argwhere(is_max):
        phi0 = np.concatenate([grid[pt], [0.0]])
        phi, ok, ismax = _polish(ext, th, phi0)
        if not ismax:
            continue
        z = np.exp(1j * phi)
        if not any(np.abs(z - z2).max() < 1e-6 for z2, _ in found):
            found.append((z, am.functional(ext, th, phi) / (d * V)))
    return found


@pytest.mark.parametrize("ext,n_grid,seeds", [((2, 2), 96, (41, 52, 54)), ((3, 2), 30, (40, 44, 45))])
def test_brute_force_grid_scan(oracle, ext, n_grid, seeds):
    """Every local maximum of F on 2x2 (double bonds, R4) and 3x2 (odd extent, R3) located by a dense phi-grid
    scan equals, as a set, what relaxation from 4096 random starts finds: F/(dV) to 1e-9 and the canonical
    configurations to 1e-5.  omega = 1.7 and omega = 1 (the paper's setting) both."""
    V = int(np.prod(ext))
    for seed in seeds:
        th = hot(ext, seed)
        brute = _brute_force_maxima(ext, th, n_grid)
        assert len(brute) >= 1
        for omega in (1.7, 1.0):
            r = oracle.relax(ext, th, seed, 4096, omega=omega, eps=1e-14, want_g=True)
            assert (r["status"] & 1).max() == 0
            c = oracle.count_copies(r["F_norm"], r["sig"], r["status"], g_canon=r["g_canon"])
            assert c["n_distinct"] == len(brute), (ext, seed, omega, c["F_rep"], [b[1] for b in brute])
            for rep in c["rep"]:
                zc = r["g_canon"][rep][:, 0] + 1j * r["g_canon"][rep][:, 1]
                match = [b for b in brute if np.abs(zc - b[0]).max() < 1e-5]
                assert len(match) == 1
                assert abs(match[0][1] - r["F_norm"][rep]) < 1e-9
                lam, region = oracle.fp_lambda1(ext, th, r["g_canon"][rep])
                assert region == 1 and lam > 0


# ------------------------------------------------------------------------------------------------ P3
def _twist(ext, k):
    x = am.coords(ext)
    return 2 * np.pi * sum(k[mu] * x[:, mu] / ext[mu] for mu in range(len(ext)))


def test_cold_orbit_bound_and_trivial_copy(oracle):
    """Cold orbit: F <= dV with equality at constant g; lambda_1(trivial) = 2(1 - cos 2pi/N)."""
    for ext in [(4, 4), (6, 6), (4, 4, 4), (4, 4, 4, 4), (3, 2), (5, 5)]:
        V, d = int(np.prod(ext)), len(ext)
        th = synth.cold_links(ext)
        F, vt, D = oracle.measure(ext, th, am.to_g(np.full(V, 0.7)))
        assert abs(F - d * V) < 1e-12 * V and vt < 1e-30
        for s in range(5):
            assert oracle.measure(ext, th, oracle.start(V, 1, s))[0] <= d * V
        lam, region = oracle.fp_lambda1(ext, th, am.to_g(np.zeros(V)))
        nmax = max(ext)
        lam_exact = 2 * (1 - np.cos(2 * np.pi / nmax)) * (2 if nmax == 2 else 1)
        assert abs(lam - lam_exact) < 1e-12 and region == 1
    # relaxation on the 4x4 cold orbit finds exactly the trivial copy
    r = oracle.relax((4, 4), synth.cold_links((4, 4)), 3, 512)
    c = oracle.count_copies(r["F_norm"], r["sig"], r["status"])
    assert c["n_distinct"] == 1 and abs(c["F_rep"][0] - 1.0) < 1e-12


def test_cold_orbit_twist_copies(oracle):
    """Twists g_x = exp(2 pi i k.x/N) on the cold orbit are stationary with F/(dV) = (1/d) sum_mu cos(2 pi k_mu/N)
    and FP spectrum sum_mu 2 c_mu (1 - cos 2 pi m_mu / N): closed-form lambda_1 and region 1 / 2 / 0."""
    cases = [((5, 5), (1, 0)), ((5, 5), (1, 1)), ((6, 6), (1, 0)), ((6, 6), (2, 0)), ((4, 4), (1, 0)),
             ((6, 6, 6), (1, 0, 1)), ((8, 8), (3, 1)), ((6, 6), (2, 2))]
    for ext, k in cases:
        V, d, N = int(np.prod(ext)), len(ext), ext[0]
        th = synth.cold_links(ext)
        g = am.to_g(_twist(ext, k))
        F, vt, D = oracle.measure(ext, th, g)
        c = np.array([np.cos(2 * np.pi * km / N) for km in k])
        assert abs(F / (d * V) - c.mean()) < 1e-13 and vt < 1e-28
        spec = [sum(2 * c[mu] * (1 - np.cos(2 * np.pi * m[mu] / N)) for mu in range(d))
                for m in np.ndindex(*ext) if any(m)]
        lam, region = oracle.fp_lambda1(ext, th, g)
        assert abs(lam - min(spec)) < 1e-11
        expect = 1 if min(spec) > 1e-8 else (2 if abs(min(spec)) <= 1e-8 else 0)
        assert region == expect
    # 5x5: relaxation finds the trivial copy and the four single twists k = (+-1,0),(0,+-1), F/(dV) = (1+cos 72deg)/2
    ext = (5, 5)
    r = oracle.relax(ext, synth.cold_links(ext), 9, 4096, want_g=True)
    cc = oracle.count_copies(r["F_norm"], r["sig"], r["status"], g_canon=r["g_canon"])
    vals = np.sort(cc["F_rep"])
    assert cc["n_distinct"] == 5
    assert np.abs(vals[:4] - (1 + np.cos(2 * np.pi / 5)) / 2).max() < 1e-12 and abs(vals[4] - 1) < 1e-12
    # the four twists have EQUAL F and are separated only by the configuration / signature test
    assert cc["margins"]["min_between_sig"] > 1e-3


# ------------------------------------------------------------------------------------------------ P4
@pytest.mark.parametrize("ext", [(4, 4), (8, 8), (4, 4, 4), (4, 4, 4, 4), (3, 3, 3, 3), (6, 3)])
def test_pure_gauge_orbit(oracle, ext):
    """theta_{i,mu} = eta_{i+mu} - eta_i: every plaquette trivial; global maximum F = dV exactly at g~ = h~
    (h = exp(i eta)), found by relaxation; lambda_1 = 2 (1 - cos 2 pi / N_max)."""
    V, d = int(np.prod(ext)), len(ext)
    eta = rand_phi(V, 51)
    th = synth.gauge_transform_links(ext, synth.cold_links(ext), -eta)   # theta = -eta_i + eta_{i+mu}
    assert np.abs(am.plaquettes(ext, th)).max() < 1e-13
    r = oracle.relax(ext, th, 51, 64, want_g=True)
    best = int(np.argmax(r["F_norm"]))
    assert abs(r["F_norm"][best] - 1.0) < 1e-12
    hz = np.exp(1j * (eta - eta[-1]))
    gz = r["g_canon"][best][:, 0] + 1j * r["g_canon"][best][:, 1]
    assert np.abs(gz - hz).max() < 1e-5
    lam, region = oracle.fp_lambda1(ext, th, r["g_canon"][best])
    assert abs(lam - 2 * (1 - np.cos(2 * np.pi / max(ext)))) < 1e-9 and region == 1
    assert (r["F_norm"] <= 1 + 1e-14).all()


# ------------------------------------------------------------------------------------------------ P5
@pytest.mark.parametrize("ext", [(4, 4), (3, 2), (4, 4, 4), (2, 2, 2, 2), (3, 3, 3, 3)])
def test_gauge_covariance(oracle, ext):
    """U' = h U h*_{i+mu}, g' = g h*  =>  identical F and g'(t) = g(t) h* along the whole trajectory; plaquette
    angles are gauge invariant mod 2 pi."""
    V = int(np.prod(ext))
    th = hot(ext, 61)
    eta = rand_phi(V, 62)
    th2 = synth.gauge_transform_links(ext, th, eta)
    assert np.abs(np.angle(np.exp(1j * (am.plaquettes(ext, th) - am.plaquettes(ext, th2))))).max() < 1e-12
    phi0 = rand_phi(V, 63)
    g, g2 = am.to_g(phi0), am.to_g(phi0 - eta)
    for t in range(12):
        g, _ = oracle.sweeps(ext, th, g, 1.7)
        g2, _ = oracle.sweeps(ext, th2, g2, 1.7)
        F1, F2 = oracle.measure(ext, th, g)[0], oracle.measure(ext, th2, g2)[0]
        assert abs(F1 - F2) < 1e-11
        z = (g[:, 0] + 1j * g[:, 1]) * np.exp(-1j * eta)
        assert np.abs(z - (g2[:, 0] + 1j * g2[:, 1])).max() < 1e-11
    # the transformed links of the found g have the plaquettes of the original links
    phi = am.to_phi(g)
    tg = am.gauged_angles(ext, th, phi).reshape(-1)
    assert np.abs(np.angle(np.exp(1j * (am.plaquettes(ext, tg) - am.plaquettes(ext, th))))).max() < 1e-12
    # independent starts on the two orbits: same multiset of copies
    if V <= 16:
        a = oracle.relax(ext, th, 5, 2048)
        b = oracle.relax(ext, th2, 6, 2048)
        ca = oracle.count_copies(a["F_norm"], a["sig"], a["status"])
        cb = oracle.count_copies(b["F_norm"], b["sig"], b["status"])
        assert ca["n_distinct"] == cb["n_distinct"]
        assert np.abs(np.sort(ca["F_rep"]) - np.sort(cb["F_rep"])).max() < 1e-10


# ------------------------------------------------------------------------------------------------ P6
@pytest.mark.parametrize("N", [5, 8, 12])
def test_one_dimensional_ring_closed_form(oracle, N):
    """1-D periodic ring (solved analytically): the copies in the first region are the uniform
    solutions theta^g = alpha_k = (Phi + 2 pi k)/N with cos alpha_k > 0, Phi = sum theta;
    F/V = cos alpha_k, lambda_1 = 2 cos alpha_k (1 - cos 2 pi/N)."""
    ext = (N,)
    th = hot(ext, 70 + N)
    Phi = th.sum()
    alphas = [(Phi + 2 * np.pi * k) / N for k in range(-N, N)]
    predicted = sorted({round(np.cos(a), 12) for a in alphas if np.cos(a) > 1e-9})
    r = oracle.relax(ext, th, 7, 4096, eps=1e-16, want_g=True)
    c = oracle.count_copies(r["F_norm"], r["sig"], r["status"], g_canon=r["g_canon"])
    assert c["n_distinct"] >= 2
    for rep, Fr in zip(c["rep"], c["F_rep"]):
        assert min(abs(Fr - p) for p in predicted) < 1e-9          # found subset of predicted
        tg = am.gauged_angles(ext, th, am.to_phi(r["g_canon"][rep])).reshape(-1)
        assert np.abs(np.angle(np.exp(1j * (tg - tg[0])))).max() < 1e-6   # uniform transformed links
        lam, region = oracle.fp_lambda1(ext, th, r["g_canon"][rep])
        assert abs(lam - 2 * Fr * (1 - np.cos(2 * np.pi / N))) < 1e-8 and region == 1
    assert abs(max(c["F_rep"]) - max(predicted)) < 1e-9            # the global maximum is found


# ------------------------------------------------------------------------------------------- P7 / P8
@pytest.mark.parametrize("ext", [(4, 4), (3, 2), (2, 2), (4, 4, 4), (3, 3, 3, 3), (4, 4, 4, 4), (6, 2, 5)])
@pytest.mark.parametrize("omega", [1.0, 1.7, 1.95])
def test_sweep_invariants(oracle, ext, omega):
    """F non-decreasing under every sweep for omega in [1,2) (local maximisation of Eq. 4); sum_i Delta_i = 0
    (lattice divergence of a periodic field); |g_i| = 1; at convergence Delta -> 0 and F = 1/2 sum_i |w_i| (P8)."""
    V, d = int(np.prod(ext)), len(ext)
    th = hot(ext, 81)
    g = oracle.start(V, 81, 3)
    Fold = oracle.measure(ext, th, g)[0]
    for t in range(40):
        g, _ = oracle.sweeps(ext, th, g, omega)
        F, vt, D = oracle.measure(ext, th, g)
        assert F >= Fold - 1e-12
        assert abs(D.sum()) < 1e-13 * V
        assert np.abs(np.hypot(g[:, 0], g[:, 1]) - 1).max() < 1e-15
        assert F <= d * V
        Fold = F
    g, _ = oracle.sweeps(ext, th, g, omega, 3000)
    F, vt, D = oracle.measure(ext, th, g)
    assert vt < 1e-24
    w = oracle.neighbour_sums(ext, th, g)
    assert abs(F - 0.5 * np.hypot(w[:, 0], w[:, 1]).sum()) < 1e-11 * V


def test_local_update_maximises_eq4(oracle):
    """omega = 1: after a sweep, every site of the LAST updated parity sits at its local optimum, Delta_i = 0
    (g_i equals the phase of K_i*), and no other value of g_i gives a larger F."""
    ext = (4, 4, 4)
    V = 64
    th = hot(ext, 91)
    g, _ = oracle.sweeps(ext, th, oracle.start(V, 91, 0), 1.0)
    F, _, D = oracle.measure(ext, th, g)
    odd = am.coords(ext).sum(1) % 2 == 1
    assert np.abs(D[odd]).max() < 1e-14 and np.abs(D[~odd]).max() > 1e-3
    rng = np.random.default_rng(1)
    for i in np.nonzero(odd)[0][:8]:
        for _ in range(20):
            g2 = g.copy()
            a = rng.uniform(-np.pi, np.pi)
            g2[i] = (np.cos(a), np.sin(a))
            assert oracle.measure(ext, th, g2)[0] <= F + 1e-12


def test_odd_extent_reading_r3(oracle):
    """R3: the oracle's sequential in-place order inside a parity class equals 2(d'+1) CONCURRENT level phases
    (what a GPU runs), and differs at O(1) from a naive concurrent two-colour update on odd extents."""
    for ext in [(3, 2), (3, 3), (5, 3, 2), (3, 3, 3, 3), (4, 4), (4, 6, 2)]:
        V = int(np.prod(ext))
        th = hot(ext, 95)
        g = oracle.start(V, 95, 1)
        a, b, c = g.copy(), g.copy(), g.copy()
        for t in range(10):
            a, _ = oracle.sweeps(ext, th, a, 1.7)
            b = am.phased_sweep(ext, th, b, 1.7)
            c = am.phased_sweep(ext, th, c, 1.7, naive_two_colour=True)
        assert np.abs(a - b).max() < 1e-12
        if any(n % 2 for n in ext):
            assert np.abs(a - c).max() > 1e-3
        else:
            assert np.abs(a - c).max() < 1e-12


def test_stop_rule_and_status(oracle):
    """O4: sweeps[k] is the first multiple of check_every with vartheta < eps; max_sweeps sets status bit0."""
    ext = (4, 4)
    th = hot(ext, 1)
    r1 = oracle.relax(ext, th, 1, 64, check_every=1)
    r4 = oracle.relax(ext, th, 1, 64, check_every=4)
    assert (r4["sweeps"] == 4 * ((r1["sweeps"] + 3) // 4)).all()
    assert (r1["vt_stop"] < 1e-13).all() and (r1["vt_prev"] >= 1e-13).all()
    for k in range(4):                                   # replay start k by hand
        g = oracle.start(16, 1, k)
        g, _ = oracle.sweeps(ext, th, g, 1.7, int(r1["sweeps"][k]) - 1)
        assert oracle.measure(ext, th, g)[1] >= 1e-13
        g, _ = oracle.sweeps(ext, th, g, 1.7, 1)
        F, vt, _ = oracle.measure(ext, th, g)
        assert vt < 1e-13 and vt == r1["vt_stop"][k] and abs(F / 32 - r1["F_norm"][k]) < 1e-15
    rs = oracle.relax(ext, th, 1, 64, max_sweeps=10)
    assert (rs["status"] & 1).all() and (rs["sweeps"] == 10).all()
    c = oracle.count_copies(rs["F_norm"], rs["sig"], rs["status"])
    assert c["n_distinct"] == 0 and (c["copy_id"] == -1).all()
    # explicit start ids reproduce the same starts
    ids = np.array([5, 3, 60, 3], dtype=np.uint64)
    ri = oracle.relax(ext, th, 1, 0, start_ids=ids)
    assert (ri["F_norm"] == r1["F_norm"][[5, 3, 60, 3]]).all() and (ri["sweeps"] == r1["sweeps"][[5, 3, 60, 3]]).all()
    # degenerate |w| = 0: cold 2x2 with a staggered start has every neighbour sum zero -> sites left alone (R6)
    g0 = np.array([[1.0, 0.0], [0.0, 1.0], [0.0, -1.0], [-1.0, 0.0]])       # w_i = 2(g_right + g_up) = 0 exactly
    th0 = synth.cold_links((2, 2))
    assert np.abs(oracle.neighbour_sums((2, 2), th0, g0)).max() == 0
    g1, skipped = oracle.sweeps((2, 2), th0, g0, 1.7)
    assert skipped and (g1 == g0).all()
    g1, skipped = oracle.sweeps((4, 4), hot((4, 4), 1), oracle.start(16, 1, 0), 1.7)
    assert not skipped


# ------------------------------------------------------------------------------------------------ P9
def test_fp_inertia_matches_eigenvalue_sign(oracle):
    """Two independent routes: LDL^T inertia of the grounded FP matrix (row/column V-1 deleted; its number of
    negative pivots is the Morse index) vs the sign of lambda_1; positive weights => positive semidefinite."""
    for ext, seed in [((4, 4), 1), ((4, 4, 4), 3), ((3, 3, 3, 3), 12), ((6, 6), 5)]:
        V = int(np.prod(ext))
        th = hot(ext, seed)
        r = oracle.relax(ext, th, seed, 16, want_g=True)
        for k in range(16):
            fields = [r["g_canon"][k], oracle.start(V, seed, 100 + k)]   # a converged copy and a random field
            for g in fields:
                M = oracle.fp_matrix(ext, th, g)
                assert np.abs(M.sum(1)).max() < 1e-13 and np.abs(M - M.T).max() == 0     # M 1 = 0, symmetric
                assert np.linalg.eigvalsh(M)[-1] <= 4 * len(ext) + 1e-12                 # Gershgorin
                lam, region = oracle.fp_lambda1(ext, th, g)
                _, Dm, _ = scipy.linalg.ldl(M[:-1, :-1])
                n_neg = int((np.linalg.eigvalsh(Dm) < 0).sum())
                assert (n_neg == 0) == (lam > 0)
                ev = np.linalg.eigvalsh(M)
                assert abs(lam - (ev[1] if lam > 0 else ev[0])) < 1e-10
            lam, region = oracle.fp_lambda1(ext, th, r["g_canon"][k])
            assert region == 1                                   # relaxation ends in minima of F_paper (L50)
            c = np.cos(am.gauged_angles(ext, th, am.to_phi(r["g_canon"][k])))
            if (c > 0).all():
                assert lam > 0


# ----------------------------------------------------------------------------------------------- P11
def test_ensemble_statistics_match_paper_tables(oracle):
    """Tab. I / Tab. III: average number of minima and average global-minimum value
    x = 1 - F/(dV) over hot orbits at omega = 1.  Our orbits (other seeds, fewer starts) must agree within
    4 combined standard errors for x and lie in a generous band for the counts (ours are lower bounds with far
    fewer starts than the paper's 4 mebisamples)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "paper_tables.txt")) if l.strip() and not l.startswith("#")]
    plan = {(2, 2): (100, 256), (2, 4): (100, 1024), (2, 6): (40, 2048), (3, 2): (100, 256), (3, 4): (20, 2048),
            (4, 2): (100, 512)}
    for row in rows:
        d, N = int(row[0]), int(row[1])
        n_paper, avg_n, std_n, avg_x, std_x = int(row[2]), *map(float, row[3:7])
        n_orb, n_starts = plan[(d, N)]
        ext = (N,) * d
        xs, ns = [], []
        for seed in range(1000, 1000 + n_orb):
            r = oracle.relax(ext, hot(ext, seed), seed, n_starts, omega=1.0)
            c = oracle.count_copies(r["F_norm"], r["sig"], r["status"])
            xs.append(1 - c["F_rep"].max())
            ns.append(c["n_distinct"])
        se = np.hypot(std_x / np.sqrt(n_paper), np.std(xs) / np.sqrt(n_orb))
        assert abs(np.mean(xs) - avg_x) < 4 * se, (d, N, np.mean(xs), avg_x, se)
        assert abs(np.std(xs) - std_x) < 0.5 * std_x
        if (d, N) in [(2, 2), (2, 4), (3, 2), (4, 2)]:           # saturated with our start counts
            se_n = np.hypot(std_n / np.sqrt(n_paper), np.std(ns) / np.sqrt(n_orb))
            assert abs(np.mean(ns) - avg_n) < 4 * se_n + 0.15 * avg_n, (d, N, np.mean(ns), avg_n)
        else:
            assert 0.2 * avg_n < np.mean(ns) <= 1.3 * avg_n


# ----------------------------------------------------------------------------------------------- P12
def test_omega_changes_basins_not_copies(oracle):
    """omega only changes which basin a start falls into: on saturated small orbits the SET of copies found with
    omega = 1 (the paper's algorithm) equals the set found with omega = 1.7."""
    for ext, seed in [((4, 4), 1), ((2, 2, 2, 2), 12), ((4, 4), 7)]:
        th = hot(ext, seed)
        sets = []
        for omega in (1.0, 1.7):
            r = oracle.relax(ext, th, seed, 8192, omega=omega)
            c = oracle.count_copies(r["F_norm"], r["sig"], r["status"])
            sets.append(np.sort(c["F_rep"]))
        assert len(sets[0]) == len(sets[1]) and np.abs(sets[0] - sets[1]).max() < 1e-10


# ------------------------------------------------------------------------------------------- O6 / O8
def test_canonical_form_and_signature(oracle):
    V = 81
    g = oracle.start(V, 2, 2)
    gc, sig = oracle.canonicalise(g)
    assert abs(gc[-1, 0] - 1) < 1e-15 and abs(gc[-1, 1]) < 1e-15              # angle at site (N,..,N) is zero (L65)
    z, zc = g[:, 0] + 1j * g[:, 1], gc[:, 0] + 1j * gc[:, 1]
    assert np.abs(zc - z * np.conj(z[-1])).max() < 1e-15
    rot = z * np.exp(0.83j)                                                   # global phase drops out
    gc2, sig2 = oracle.canonicalise(np.stack([rot.real, rot.imag], 1))
    assert np.abs(gc2 - gc).max() < 1e-15 and np.abs(sig2 - sig).max() < 1e-15
    a, b = oracle.signature_signs(V)
    assert set(np.unique(a)) == {-1.0, 1.0} and set(np.unique(b)) == {-1.0, 1.0}
    assert abs(a.mean()) < 0.2 and abs(b.mean()) < 0.2
    assert np.abs(sig - (a * gc[:, 0] + b * gc[:, 1]).mean(axis=1)).max() < 1e-15
    w = synth.philox4x32_10(np.arange(V, dtype=np.uint64), 2, 0, 1, 0x51, 0)   # sign bits from the numpy Philox
    assert ((w[0] & np.uint64(1)) * 2.0 - 1 == a[2]).all() and ((w[1] & np.uint64(1)) * 2.0 - 1 == b[2]).all()


def test_count_copies_hand_made_records(oracle):
    """O8/O9 on records whose grouping is known by construction."""
    sA, sB, sC = np.array([.1, .2, .3, .4]), np.array([.1, .2, .3, .4]) + 0.01, np.array([-.3, .2, .1, 0])
    F = np.array([0.50, 0.70, 0.50 + 2e-11, 0.50, 0.70 + 5e-11, 0.9, 0.50 - 3e-11, 0.70])
    sig = np.array([sA, sC, sA + 1e-6, sB, sC - 2e-5, sA, sB + 1e-5, sA])
    status = np.array([0, 0, 0, 0, 0, 1, 0, 2], dtype=np.uint8)              # record 5 not converged; bit1 is harmless
    c = oracle.count_copies(F, sig, status, nbins=10)
    # discovery order: copy 0 = {0,2} (F .5, sA), copy 1 = {1,4} (F .7, sC), copy 2 = {3,6} (F .5, sB), copy 3 = {7}
    assert c["copy_id"].tolist() == [0, 1, 0, 2, 1, -1, 2, 3]
    assert c["n_distinct"] == 4 and c["rep"].tolist() == [0, 1, 3, 7] and c["multiplicity"].tolist() == [2, 2, 2, 1]
    assert c["hist"].tolist() == [0, 0, 0, 0, 0, 4, 0, 3, 0, 0]
    # chained run: gaps of 0.8 tol_F each are one run even though its ends are 1.6 tol_F apart
    F2 = np.array([0.3, 0.3 + 0.8e-10, 0.3 + 1.6e-10, 0.3 + 2.8e-10])
    c2 = oracle.count_copies(F2, np.tile(sA, (4, 1)), np.zeros(4, np.uint8))
    assert c2["copy_id"].tolist() == [0, 0, 0, 1]
    c0 = oracle.count_copies(np.zeros(0), np.zeros((0, 4)), np.zeros(0, np.uint8), nbins=4)
    assert c0["n_distinct"] == 0 and c0["hist"].tolist() == [0, 0, 0, 0]


def test_discovery_curve_and_paper_count_pins(oracle):
    """SURVEY 8(f)-1.  Discovery curve (Figs. 1-3) and the paper's floor(x*1e8) count (L133-135) on
    records whose answers are known by construction, plus the properties that hold for any input."""
    # copies first seen at positions 0, 1, 2, 5, 8, 1000: among the first 1, 2, 4, 8, 16, ... samples
    rep = np.array([0, 1, 2, 5, 8, 1000])
    assert oracle.discovery_curve(rep, 12).tolist() == [1, 2, 3, 4, 5, 5, 5, 5, 5, 5, 6, 6]
    assert oracle.discovery_curve(np.zeros(0, np.int64), 3).tolist() == [0, 0, 0]
    # ties to count_copies: the curve ends at n_distinct, never decreases, and curve[k] <= 2^k
    F = np.array([0.50, 0.70, 0.50 + 2e-11, 0.61, 0.70 + 5e-11, 0.9, 0.33, 0.70])
    sig = np.tile(np.array([.1, .2, .3, .4]), (8, 1))
    c = oracle.count_copies(F, sig, np.zeros(8, np.uint8))
    cur = oracle.discovery_curve(c["rep"], 5)           # copies first seen at positions 0, 1, 3, 5, 6
    assert c["rep"].tolist() == [0, 1, 3, 5, 6]
    assert cur.tolist() == [1, 2, 3, 5, 5] and cur[-1] == c["n_distinct"]
    assert (np.diff(cur) >= 0).all() and all(cur[k] <= (1 << k) for k in range(5))
    # paper count: x = 1 - F in units of 1e-8.  0.123456782 and 0.123456787 share the key 12345678; 0.123456793
    # has the next key; a non-converged record is ignored; 1 - F is formed first, as the paper defines x
    x = np.array([0.123456782, 0.123456787, 0.123456793, 0.5, 0.9])
    st = np.array([0, 0, 0, 0, 1], dtype=np.uint8)
    assert oracle.paper_count(1.0 - x, st) == 3
    assert oracle.paper_count(1.0 - x, np.zeros(5, np.uint8)) == 4
    assert oracle.paper_count(np.zeros(0), np.zeros(0, np.uint8)) == 0
    # a coarser resolution merges: at 1e-2 the keys are 12, 12, 12, 50
    assert oracle.paper_count(1.0 - x, st, scale=1e2) == 2
    # R7 in one picture: two copies 3e-9 apart in F/(dV) that the signature separates are ONE key for the paper
    Fc = np.array([0.6000000012, 0.6000000042])
    sg = np.array([[.1, .2, .3, .4], [-.3, .2, .1, 0.]])
    assert oracle.count_copies(Fc, sg, np.zeros(2, np.uint8))["n_distinct"] == 2
    assert oracle.paper_count(Fc, np.zeros(2, np.uint8)) == 1


def test_ensemble_readout_pins(oracle):
    """SURVEY 8(f)-3 read-outs on hand-made copy tables whose answers are worked out by hand (binary fractions, so
    every value below is exact in FP64)."""
    # three orbits: best F/(dV) 0.75, 0.5, 0.875 -> x_g 0.25, 0.5, 0.125; copies 3, 1, 2
    Fs = [np.array([0.5, 0.75, 0.25]), np.array([0.5]), np.array([0.875, 0.75])]
    ms = [np.array([2, 5, 1]), np.array([4]), np.array([1, 3])]
    st = oracle.ensemble_stats(Fs, n_in_region=[3, 1, 0])
    assert st["best_x"].tolist() == [0.25, 0.5, 0.125]
    assert st["n_distinct"] == (2.0, 1.0)                      # mean of 3,1,2; sqrt(((1)^2+(1)^2+0)/2) = 1
    assert st["best"][0] == 0.875 / 3 and abs(st["best"][1] - np.std([0.25, 0.5, 0.125], ddof=1)) < 1e-15
    assert st["n_in_region"][0] == 4.0 / 3 and abs(st["n_in_region"][1] - np.std([3, 1, 0], ddof=1)) < 1e-15
    assert st["used"] == 3
    # one orbit: standard deviation 0; an orbit without copies is NaN and left out of the x_g average
    assert oracle.ensemble_stats([np.array([0.5])])["n_distinct"] == (1.0, 0.0)
    s2 = oracle.ensemble_stats([np.array([0.5]), np.zeros(0)])
    assert np.isnan(s2["best_x"][1]) and s2["best"] == (0.5, 0.0) and s2["used"] == 1 and s2["n_distinct"][0] == 0.5
    # relative deviation (x_i - x_g)/x_g.  Orbit 0: x = 0.5, 0.25, 0.75 with x_g 0.25 -> dev 1, 0, 2 (weights 2, 5, 1);
    # orbit 1: dev 0 (weight 4); orbit 2: x = 0.125, 0.25 -> dev 0, 1 (weights 1, 3).  4 bins on [0, 2): width 0.5
    r = oracle.relative_deviation_hist(Fs, ms, dev_max=2.0, nbins=4)
    assert r["counts"].tolist() == [[5, 0, 2, 1], [4, 0, 0, 0], [1, 0, 3, 0]]      # dev 2 >= dev_max: last bin
    assert r["n_converged"].tolist() == [8, 4, 4] and r["used"] == 3
    assert np.allclose(r["avg"], [(5 / 8 + 1 + 1 / 4) / 3, 0, (2 / 8 + 3 / 4) / 3, (1 / 8) / 3], rtol=0, atol=1e-16)
    assert abs(r["avg"].sum() - 1.0) < 1e-15                    # fractions of samples: the average sums to one
    # the trivial orbit (F/(dV) = 1, x_g = 0) and an empty orbit are left out
    r2 = oracle.relative_deviation_hist([np.array([1.0, 0.5]), np.zeros(0), np.array([0.5, 0.25])],
                                        [np.array([3, 1]), np.zeros(0, np.int64), np.array([1, 1])], dev_max=1.0, nbins=2)
    assert r2["counts"].tolist() == [[0, 0], [0, 0], [1, 1]] and r2["used"] == 1 and r2["avg"].tolist() == [0.5, 0.5]
    # scale invariance: the same copies with every multiplicity times 64 give the same averaged distribution
    r3 = oracle.relative_deviation_hist(Fs, [64 * m for m in ms], dev_max=2.0, nbins=4)
    assert (r3["avg"] == r["avg"]).all() and (r3["counts"] == 64 * r["counts"]).all()
    # Fig. 5 ratios: 64 times the samples in every bin but the last two
    h = oracle.hist_ratio(np.array([2, 0, 5, 0, 3]), np.array([128, 0, 320, 7, 0]))
    assert h["ratio"][0] == 64.0 and np.isnan(h["ratio"][1]) and h["ratio"][2] == 64.0 and np.isinf(h["ratio"][3])
    assert h["ratio"][4] == 0.0 and h["n_only"] == (1, 1)
