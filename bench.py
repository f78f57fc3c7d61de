#!/usr/bin/env python
"""bench.py -- throughput of the u1gf hot path on B200 (contract: one JSON line on stdout from rank 0).

A "step" is one pass of the whole hot path (a2-a8) over one batch of synthetic starts of the
workload BASELINE.json's target is quoted on: config 4 = 4D 4^4, Gaussian(0.8)+gauge-transformed orbit (seed 11),
2^22 random starts, omega 1.7, eps 1e-13:
    u1gf_relax_batch -> u1gf_count_copies -> u1gf_relax_batch(start_ids = representatives, g_canon) -> u1gf_check_fp
`value` = relaxation site-updates/s = V * sum(sweeps) / step time (device-resident, CUDA events).
`e2e`   = the same through the *_host C-ABI entry points (host buffers, H2D/D2H inside the timed region).
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1403_0555_b200 import shard, synth  # noqa: E402

METRIC = "relaxation_site_updates_per_s"
UNIT = "site-updates/s"
A_D = {1: 24, 2: 32, 3: 40, 4: 48}   # algorithmic FP64 instructions per site update, 8d+16


def workload(cfg_id, orbit_idx, n_override):
    conf = synth.CONFIGS[cfg_id]
    ob = dict(conf["orbits"][orbit_idx])
    if n_override:
        ob["n_starts"] = n_override
    return conf, ob


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index):
        self.lines, self.proc, self.index = [], None, index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_leg(conf, ob, budget_s, n_first=1024):
    """The oracle as it stands on the host cores, on a bounded prefix of the workload's starts."""
    import oracle
    ext, seed = ob["extents"], ob["seed"]
    th = synth.make_theta(ob)
    V = synth.volume(ext)
    kw = dict(omega=conf["omega"], eps=conf["eps"], max_sweeps=conf["max_sweeps"])
    t0 = time.perf_counter()
    r = oracle.relax(ext, th, seed, n_first, **kw)
    t1 = time.perf_counter() - t0
    n = int(min(ob["n_starts"], max(n_first, n_first * budget_s / max(t1, 1e-3))))
    t0 = time.perf_counter()
    r = oracle.relax(ext, th, seed, n, first_start=0, **kw)
    c = oracle.count_copies(r["F_norm"], r["sig"], r["status"])
    dt = time.perf_counter() - t0
    su = float(V) * float(r["sweeps"].sum())
    return dict(value=su / dt, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                sample=f"first {n} starts of the workload ({su:.3g} site-updates, {dt:.1f} s, relax+count)",
                copies_per_s=float(((r["status"] & 1) == 0).sum()) / dt, n_distinct_in_sample=int(c["n_distinct"])), dt, su


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="u1gf", choices=["u1gf", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE config id (1..5); 4 is the metric's workload")
    ap.add_argument("--orbit", type=int, default=0, help="orbit index inside the config")
    ap.add_argument("--starts", type=int, default=0, help="override the number of starts (debugging only)")
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 force the generic kernel")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    ri = shard.rank_info_from_env()
    rank, world, local = ri.rank, ri.world, ri.local_rank
    conf, ob = workload(args.config, args.orbit, args.starts)
    ext, seed, n = ob["extents"], ob["seed"], ob["n_starts"]
    V, d = synth.volume(ext), len(ext)
    wl = f"config {args.config} orbit {args.orbit}: {conf['name']} {'x'.join(map(str, ext))} seed {seed}, {n} starts"
    config = {"workload": wl, "extents": list(ext), "starts_per_step": n, "omega": conf["omega"], "eps": conf["eps"],
              "max_sweeps": conf["max_sweeps"], "l2": "flushed between steps (256 MiB write); state is on-chip"}

    if args.impl == "reference":
        if rank != 0:
            return 0
        vals, dts = [], []
        for _ in range(args.warmup):
            oracle_leg(conf, ob, 0.5, n_first=256)
        last = None
        for _ in range(max(args.steps, 1)):
            last, dt, su = oracle_leg(conf, ob, 6.0)
            vals.append(su); dts.append(dt)
        v = sum(vals) / sum(dts)
        last["value"] = v
        print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": 0,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(dts) / len(dts),
                          "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                          "data": "synthetic", "config": config, "cpu_baseline": last,
                          "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return 0

    import torch
    from paper_1403_0555_b200 import binding as b
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    b.lib()
    th = synth.make_theta(ob)
    orbit = b.Orbit(ext, th)
    orbit.set_kernel(args.kernel)
    first, _ = shard.weak_start_range(rank, world, n)   # disjoint start ranges of the same orbit, no data-path collective
    kw = dict(omega=conf["omega"], eps=conf["eps"], max_sweeps=conf["max_sweeps"])
    nbins = 10000
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    out = ws = cws = None
    state = {}

    def step():
        nonlocal out, ws, cws
        launches = 0
        out = b.relax_batch(orbit, seed, n, first_start=first, out=out, workspace=ws, **kw)
        ws = out["workspace"]
        launches += b.last_launch_count()
        state["relax_ms"] = None
        c = b.count_copies(out["F_norm"], out["sig"], out["status"], nbins=nbins, workspace=cws)
        cws = c["workspace"]
        launches += b.last_launch_count()
        nd = int(c["n_distinct"].item())                       # the only host read inside a step (8 bytes)
        state["relax_ms"] = b.last_relax_ms()
        rep_ids = c["rep"][:nd] + first
        rr = b.relax_batch(orbit, seed, 0, start_ids=rep_ids, want_g=True, **kw)
        launches += b.last_launch_count()
        f = b.check_fp(orbit, rr["g_canon"])
        launches += b.last_launch_count()
        state.update(n_distinct=nd, c=c, f=f, launches=launches)

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
        flush.fill_(1)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    relax_ms = []
    for k in range(args.steps):
        ev[k][0].record()
        step()
        ev[k][1].record()
        relax_ms.append(state["relax_ms"])
        flush.fill_(k & 1)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = sum(a.elapsed_time(z) for a, z in ev)
    sweeps_sum = int(out["sweeps"].sum(dtype=torch.int64).item())
    conv = int((out["status"] & 1).eq(0).sum().item())
    total_ms, (sweeps_sum, conv) = shard.aggregate(total_ms, [sweeps_sum, conv], dist, device="cuda")
    ms_per_step = total_ms / args.steps
    site_updates = float(V) * float(sweeps_sum)              # per step, all ranks
    value = site_updates / (ms_per_step * 1e-3)

    # e2e: the same step through the host-buffer C-ABI entry points (H2D / D2H and allocation inside)
    e2e = None
    if not args.no_e2e:
        hb = b.host_buffers(n)   # pinned result arrays, made once: the timed region holds copies, not page faults

        def host_step():
            orb = b.Orbit(ext, th)
            orb.set_kernel(args.kernel)
            r = b.relax_batch_host(orb, seed, n, first_start=first, out=hb, **kw)
            c = b.count_copies_host(r["F_norm"], r["sig"], r["status"], nbins=nbins, out=hb)
            rr = b.relax_batch_host(orb, seed, 0, start_ids=(c["rep"] + first).astype(np.uint64), want_g=True, **kw)
            f = b.check_fp_host(orb, rr["g_canon"])
            nd = c["n_distinct"]
            h2d = th.nbytes + n * 41 + nd * 8 + nd * V * 16
            d2h = n * 45 + n * 4 + 8 + 2 * nd * 8 + nbins * 8 + nd * (45 + V * 16) + nd * 9 + 8
            orb.close()
            return float(V) * float(r["sweeps"].sum()), h2d, d2h
        host_step()
        barrier()
        t0 = time.perf_counter()
        su_e = 0.0
        reps = max(1, min(args.steps, 2))
        for _ in range(reps):
            su, h2d, d2h = host_step()
            su_e += su
        barrier()
        dt = time.perf_counter() - t0
        te = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if dist:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": su_e * world / float(te[0]), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "timing": "wall clock around the synchronous *_host calls, max over ranks"}

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0

    # roofline of the dominant kernel (the relaxation kernel): FP64 ALU bound
    peak_dfma = b.measure_fp64_peak(300.0)
    rate_rrr = b.measure_fp64_rate(1, 100.0)   # DFMA with three distinct register operands
    rate_mac = b.measure_fp64_rate(2, 100.0)   # the complex multiply-accumulate pattern of w_i
    k_ms = float(np.mean([m for m in relax_ms if m and m > 0])) if any(relax_ms) else None
    per_rank_su = site_updates / world
    achieved = per_rank_su * A_D[d] * 2.0 / (k_ms * 1e-3) / 1e12 if k_ms else None
    peak = peak_dfma * 2.0 / 1e12
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak if achieved else None, "traffic": None,
                "dfma_rate_3_register_operands": rate_rrr * 2.0 / 1e12, "dfma_rate_complex_mac": rate_mac * 2.0 / 1e12,
                "kernel": orbit.kernel_name, "kernel_ms": k_ms, "kernel_share_of_step": k_ms / ms_per_step if k_ms else None,
                "note": ("achieved = site-updates x (8d+16 = %d algorithmic FP64 instructions) x 2 flop / kernel time; "
                         "peak = 2 x DFMA/s of the in-run u1gf_measure_fp64_peak microbenchmark (kernel timed alone; constant "
                         "multiplicands); dfma_rate_* = the same unit for DFMA streams with register multiplicands, "
                         "which the register file limits to 3/4 of peak (DESIGN.md section 7.1)") % A_D[d]}
    if orbit.kernel_name.startswith("stream"):
        # the streamed kernel (large lattices) is bound by memory traffic: algorithmic bytes = one read and one write of
        # g per site update (32 B); peak = the driver's measured HBM copy bandwidth
        hbm_peak, how = 6650.0, "fallback of B200_PROFILING.md"
        try:
            with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                hbm_peak, how = float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json"
        except (OSError, KeyError, ValueError):
            pass
        gbs = per_rank_su * 32.0 / (k_ms * 1e-3) / 1e9 if k_ms else None
        roofline = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                    "frac": gbs / hbm_peak if gbs else None, "traffic": None, "peak_source": how,
                    "fp64_frac": roofline["frac"], "kernel": orbit.kernel_name, "kernel_ms": k_ms,
                    "kernel_share_of_step": k_ms / ms_per_step if k_ms else None,
                    "note": "achieved = site-updates x 32 algorithmic bytes / kernel time; fp64_frac = the same launch "
                            "against the measured FP64 peak (A_d algorithmic instructions per site update)"}
    cpu = None
    if not args.no_cpu_baseline:
        cpu, _, _ = oracle_leg(conf, ob, 10.0)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config, "clocks": clocks, "e2e": e2e, "gpu_launches": state["launches"],
            "roofline": roofline, "cpu_baseline": cpu,
            "converged_copies_per_s": conv / (ms_per_step * 1e-3), "n_distinct": state["n_distinct"],
            "n_in_first_region": int(state["f"]["n_in_region"].item()), "mean_sweeps": sweeps_sum / (n * world)}
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
