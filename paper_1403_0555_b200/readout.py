"""Read-outs on top of the C-ABI calls (argument marshalling and table assembly only; every number comes out of the
library's kernels).

bias_table -- SURVEY section 8(f)-2.  The paper runs plain relaxation because "overrelaxation decreases the convergence
time, [but] it also decreases the chance of converging to larger minima and thus introduces a bias".
The table lists, for every copy found by either run on the SAME random starts, its basin size (multiplicity) under
omega = 1 (the paper's algorithm) and under the over-relaxed omega: u1gf_relax_batch + u1gf_count_copies per omega, and
u1gf_merge_copy_tables to identify the copies of the two runs with each other (copy identity R7).
"""
from __future__ import annotations

import numpy as np

from . import binding as b


def bias_table(orbit: b.Orbit, seed: int, n_starts: int, *, omega: float = 1.7, eps: float = 1e-13,
               max_sweeps: int = 20000, first_start: int = 0):
    """Returns dict(F, x_paper, mult_omega1, mult_omega, sweeps_omega1, sweeps_omega): copies sorted by decreasing
    F/(dV) (increasing paper value x = 1 - F/(dV), i.e. smaller minima first), numpy arrays."""
    import torch
    n = int(n_starts)
    tabs, mean_sweeps = [], []
    for k, w in enumerate((1.0, omega)):
        r = b.relax_batch(orbit, seed, n, first_start=first_start, omega=w, eps=eps, max_sweeps=max_sweeps)
        c = b.count_copies(r["F_norm"], r["sig"], r["status"])
        nd = int(c["n_distinct"].item())
        rep = c["rep"][:nd]
        # run 1's entries are ordered behind run 0's, so that a merged copy takes its F from the omega = 1 run if it has it
        tabs.append((r["F_norm"][rep], r["sig"][rep], rep + k * n, c["multiplicity"][:nd].clone()))
        mean_sweeps.append(float(r["sweeps"].double().mean().item()))
    F = torch.cat([t[0] for t in tabs])
    S = torch.cat([t[1] for t in tabs])
    fs = torch.cat([t[2] for t in tabs])
    zeros0, zeros1 = torch.zeros_like(tabs[0][3]), torch.zeros_like(tabs[1][3])
    m0 = b.merge_copy_tables(F, S, fs, torch.cat([tabs[0][3], zeros1]))     # multiplicities of the omega = 1 run only
    m1 = b.merge_copy_tables(F, S, fs, torch.cat([zeros0, tabs[1][3]]))     # ... of the over-relaxed run only
    nm = int(m0["n_merged"].item())
    assert nm == int(m1["n_merged"].item())
    first = m0["first_start"][:nm]                       # entry that leads each merged copy
    # F of a merged copy = F of its leader (a start of run 0 if first < n, else of run 1)
    mid = m0["merged_id"]
    Fm = torch.zeros(nm, dtype=torch.float64, device=F.device)
    lead_mask = fs == first[mid.long()]
    Fm[mid[lead_mask].long()] = F[lead_mask]
    order = torch.argsort(Fm, descending=True)
    Fs = Fm[order].cpu().numpy()
    return dict(F=Fs, x_paper=1.0 - Fs, mult_omega1=m0["multiplicity"][:nm][order].cpu().numpy(),
                mult_omega=m1["multiplicity"][:nm][order].cpu().numpy(), sweeps_omega1=mean_sweeps[0],
                sweeps_omega=mean_sweeps[1], omega=omega, n_starts=n)


def format_bias_table(tab, top: int = 20) -> str:
    """Markdown table of the `top` largest basins plus the totals the paper's claim is about."""
    m1, mw = tab["mult_omega1"], tab["mult_omega"]
    n = tab["n_starts"]
    lines = [f"| x = 1 - F/(dV) | basin, omega = 1 | basin, omega = {tab['omega']} |", "|---|---|---|"]
    for k in np.argsort(-(m1 + mw))[:top]:
        lines.append(f"| {tab['x_paper'][k]:.9f} | {int(m1[k])} | {int(mw[k])} |")
    both = int(((m1 > 0) & (mw > 0)).sum())
    lines.append("")
    lines.append(f"copies found: omega = 1: {int((m1 > 0).sum())}, omega = {tab['omega']}: {int((mw > 0).sum())}, by both: {both}; "
                 f"mean sweeps {tab['sweeps_omega1']:.1f} vs {tab['sweeps_omega']:.1f}; "
                 f"mean x over starts {float((tab['x_paper'] * m1).sum() / n):.6f} vs {float((tab['x_paper'] * mw).sum() / n):.6f}")
    return "\n".join(lines)


if __name__ == "__main__":
    # python -m paper_1403_0555_b200.readout [config] [orbit] [n_starts]: the bias table of one BASELINE orbit as markdown
    import sys
    from . import synth
    cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 3
    oi = int(sys.argv[2]) if len(sys.argv) > 2 else 0
    conf = synth.CONFIGS[cfg]
    ob = conf["orbits"][oi]
    n = int(sys.argv[3]) if len(sys.argv) > 3 else ob["n_starts"]
    orbit = b.Orbit(ob["extents"], synth.make_theta(ob))
    tab = bias_table(orbit, ob["seed"], n, omega=conf["omega"], eps=conf["eps"], max_sweeps=conf["max_sweeps"])
    print(f"config {cfg} orbit {oi}: {'x'.join(map(str, ob['extents']))} seed {ob['seed']}, {n} starts, eps {conf['eps']}, kernel {orbit.kernel_name}\n")
    print(format_bias_table(tab, top=16))
