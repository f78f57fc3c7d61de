"""Every start of the BASELINE configs against the oracle (north_star: "identical start-to-copy assignment and
distinct-copy counts (bit-exact integer output) ... on all five configs"; PAPER.md:L129-135 sort and count, L149).

The other GPU modules compare full-size launches with the oracle on samples; here nothing is sampled.  Each case runs
the launch bench.py times (u1gf_relax_batch on all starts of the orbit, then u1gf_count_copies with the 1e-4 bins of
PAPER.md:L167) and the oracle on the same starts -- oracle.relax on all host cores, then oracle.count_copies -- and
compares EVERY entry of every output: sweeps, status, copy_id, n_distinct, rep, multiplicity, hist bit for bit,
F/(dV) within 1e-10, the signature within 1e-7.

Compared in full: config 2 (8x8, 2^20 starts), all 8 orbits of config 3 (4^3, 2^20 each), config 4 (4^4, 2^22),
config 5 at 2^4, 3^4, 4^4 (2^20 each) and 8^4 (2^16).  6^4 of config 5 is compared on its first 2^17 of 2^20 starts:
the oracle needs about 4 minutes for the full orbit on 16 cores; the launch is the TMA-staged kernel either way.
Config 1 is compared in full in test_gpu_parity.py.

Cost, measured on the GPU box (16 host cores): 274 s for the module, nearly all of it oracle.relax (80 s config 4, 76 s
8^4, 30 s 6^4, 27 s hot 4^4, 4 s per 4^3 orbit); oracle.count_copies, a Python loop over the F-runs, takes 2.3 s on the
hot 4^4 orbit (393047 copies) and well under a second elsewhere; the GPU side is about 2 s in all.  The module sorts
late on purpose, so these minutes come after the quick parity tests; tests/test_zz_no_alloc.py stays last.
"""
import time

import numpy as np
import pytest

from paper_1403_0555_b200 import synth

pytestmark = pytest.mark.gpu

TOL_F = 1e-10
TOL_G = 1e-7

#        cfg, orbit index, number of starts compared (None = the config's full count)
CASES = ([(2, 0, None)] + [(3, k, None) for k in range(8)] + [(4, 0, None)] +
         [(5, 0, None), (5, 1, None), (5, 2, None), (5, 3, 1 << 17), (5, 4, None)])


@pytest.fixture(scope="module")
def b():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1403_0555_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("cfg,orbit_idx,n_cmp", CASES)
def test_every_start_of_the_config_matches_the_oracle(b, oracle, cfg, orbit_idx, n_cmp):
    conf = synth.CONFIGS[cfg]
    ob = conf["orbits"][orbit_idx]
    ext, seed = ob["extents"], ob["seed"]
    n = ob["n_starts"] if n_cmp is None else n_cmp
    th = synth.make_theta(ob)
    kw = dict(omega=conf["omega"], eps=conf["eps"], max_sweeps=conf["max_sweeps"])
    orbit = b.Orbit(ext, th)
    r = b.relax_batch(orbit, seed, n, **kw)
    c = b.count_copies(r["F_norm"], r["sig"], r["status"], nbins=10000)
    g = {k: r[k].cpu().numpy() for k in ("F_norm", "sweeps", "status", "sig")}
    nd = int(c["n_distinct"].item())
    gc = dict(copy_id=c["copy_id"].cpu().numpy(), rep=c["rep"].cpu().numpy()[:nd],
              multiplicity=c["multiplicity"].cpu().numpy()[:nd], hist=c["hist"].cpu().numpy())
    del r, c

    t0 = time.time()
    o = oracle.relax(ext, th, seed, n, **kw)
    t1 = time.time()
    oc = oracle.count_copies(o["F_norm"], o["sig"], o["status"], nbins=10000)
    t2 = time.time()
    print(f"\n{conf['name']} orbit {orbit_idx} {ext} {n} starts ({orbit.kernel_name}): oracle relax {t1 - t0:.1f} s on "
          f"{oracle.num_threads()} threads, oracle count {t2 - t1:.1f} s, n_distinct {oc['n_distinct']}")

    bad = np.nonzero(o["sweeps"] != g["sweeps"])[0]
    assert bad.size == 0, (f"sweeps differ at starts {bad[:8]}: oracle {o['sweeps'][bad[:8]]} gpu {g['sweeps'][bad[:8]]}; "
                           f"oracle vartheta at its stop {o['vt_stop'][bad[:8]]}, one test earlier {o['vt_prev'][bad[:8]]}")
    assert (o["status"] == g["status"]).all()
    assert np.abs(o["F_norm"] - g["F_norm"]).max() < TOL_F
    assert np.abs(o["sig"] - g["sig"].reshape(-1, 4)).max() < TOL_G
    assert nd == oc["n_distinct"]
    assert (gc["copy_id"] == oc["copy_id"]).all()
    assert (gc["rep"] == oc["rep"]).all()
    assert (gc["multiplicity"] == oc["multiplicity"]).all() and int(gc["multiplicity"].sum()) == int((g["status"] & 1 == 0).sum())
    assert (gc["hist"] == oc["hist"]).all()
