#!/usr/bin/env python
"""bench.py -- throughput of the u1gf hot path on B200 (contract: one JSON line on stdout from rank 0).

A "step" is one pass of the whole hot path (a2-a8) over one batch of synthetic starts of the
workload BASELINE.json's target is quoted on: config 4 = 4D 4^4, Gaussian(0.8)+gauge-transformed orbit (seed 11),
2^22 random starts, omega 1.7, eps 1e-13:
    u1gf_relax_batch -> u1gf_count_copies -> u1gf_relax_batch(start_ids = representatives, g_canon) -> u1gf_check_fp
(on hot orbits, where most starts are their own copy, the fields of all starts are written in the first pass instead
and u1gf_check_fp picks the representatives by index: no second relaxation).
`value` = relaxation site-updates/s = V * sum(sweeps) / step time (device-resident, CUDA events).
`e2e`   = the same through u1gf_pipeline_host (host result buffers, D2H inside the timed region; the method's only
          host input is the link field, handed to u1gf_create_orbit inside the timed region too).
`configs` = the other BASELINE configs (1, 2, 3 as one ensemble launch, every size of 5), each timed the same way
          with fewer repetitions, so that one driver-visible run records all five (`--no-all-configs` skips them).
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
FP64_LANES_PER_SM = 64               # B200: the DMMA probe and 148 x 64 x clock agree


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
                copies_per_s=float(((r["status"] & 1) == 0).sum()) / dt, n_distinct_in_sample=int(c["n_distinct"]),
                sample_starts=n), dt, su


class Pipeline:
    """One BASELINE workload on the device: buffers made once, `step()` = the whole hot path."""

    def __init__(self, b, torch, conf, ob, first, kernel=0, nbins=10000):
        self.b, self.torch, self.conf = b, torch, conf
        self.ext, self.seed, self.n, self.first = ob["extents"], ob["seed"], ob["n_starts"], first
        self.V, self.d = synth.volume(self.ext), len(self.ext)
        self.theta = synth.make_theta(ob)
        self.orbit = b.Orbit(self.ext, self.theta)
        self.orbit.set_kernel(kernel)
        self.kw = dict(omega=conf["omega"], eps=conf["eps"], max_sweeps=conf["max_sweeps"])
        self.nbins = nbins
        self.out = self.ws = self.cws = None
        self.store_g = False          # decided after the first step: see step()
        self.ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
        self.fev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
        self.state = {}

    def step(self):
        b, torch = self.b, self.torch
        launches = 0
        if self.store_g and (self.out is None or self.out.get("g_canon") is None):
            self.out = None
        self.ev[0].record()           # the relaxation kernel, on the stream it is launched on (torch's current stream)
        self.out = b.relax_batch(self.orbit, self.seed, self.n, first_start=self.first, out=self.out, workspace=self.ws,
                                 want_g=self.store_g, **self.kw)
        self.ev[1].record()
        self.ws = self.out["workspace"]
        launches += b.last_launch_count()
        c = b.count_copies(self.out["F_norm"], self.out["sig"], self.out["status"], nbins=self.nbins, workspace=self.cws)
        self.cws = c["workspace"]
        launches += b.last_launch_count()
        nd = int(c["n_distinct"].item())                       # the only host read inside a step (8 bytes)
        self.fev[0].record()
        if self.store_g:
            f = b.check_fp(self.orbit, self.out["g_canon"], index=c["rep"][:nd], want_steps=True)
            launches += b.last_launch_count()
        else:
            rr = b.relax_batch(self.orbit, self.seed, 0, start_ids=c["rep"][:nd] + self.first, want_g=True, **self.kw)
            launches += b.last_launch_count()
            f = b.check_fp(self.orbit, rr["g_canon"], want_steps=True)
            launches += b.last_launch_count()
        self.fev[1].record()
        # hot orbits (most starts are their own copy): write the fields of all starts in the first pass from now on,
        # if they fit a quarter of the device memory -- no second relaxation of n_distinct ~ n representatives
        total_mem = torch.cuda.get_device_properties(0).total_memory
        self.store_g = nd > self.n // 4 and self.n * self.V * 16 <= total_mem // 4
        self.state.update(n_distinct=nd, c=c, f=f, launches=launches)

    def summary(self, relax_ms, fp_ms, step_ms, peak_dfma, sm_clock_mhz, sms, hbm_peak):
        torch = self.torch
        out, st = self.out, self.state
        sweeps_sum = int(out["sweeps"].sum(dtype=torch.int64).item())
        conv = int((out["status"] & 1).eq(0).sum().item())
        su = float(self.V) * float(sweeps_sum)
        nd = st["n_distinct"]
        reg = st["f"]["region"]
        exc = torch.nonzero(reg != 1).flatten()
        exc_starts = (st["c"]["rep"][:nd][exc] + self.first).cpu().tolist()
        fp64 = su * A_D[self.d] * 2.0 / (relax_ms * 1e-3) / 1e12
        peak = peak_dfma * 2.0 / 1e12
        pipe = sms * FP64_LANES_PER_SM * sm_clock_mhz * 1e6 * 2.0 / 1e12
        name = self.orbit.kernel_name
        roof = {"bound": "alu", "achieved": fp64, "peak": peak, "unit": "TFLOP/s", "frac": fp64 / peak,
                "frac_of_fp64_pipe": fp64 / pipe, "fp64_pipe_peak": pipe, "traffic": None}
        if name.startswith("stream") or name.startswith("tma_stream"):
            # 32 B of HBM per site update (g read + written once per sweep).  The checkerboard as built moves
            # 48 B (the rows of a parity are read twice per sweep: as neighbours and as the site itself), DESIGN.md 7.4
            gbs = su * 32.0 / (relax_ms * 1e-3) / 1e9
            roof = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                    "frac_at_48_bytes_moved": gbs * 1.5 / hbm_peak, "fp64_frac": fp64 / peak, "traffic": None}
        roof.update(kernel=name, kernel_ms=relax_ms, kernel_share_of_step=relax_ms / step_ms)
        # a7: (2d+1) FP64 FMAs per site and Lanczos step (the mat-vec); first_region_ms also holds the
        # re-relaxation of the representatives where the fields of all starts were not kept
        steps = st["f"]["steps"]
        lz_steps = int(steps.sum(dtype=torch.int64).item()) if steps is not None and nd else 0
        lz_fma = float(lz_steps) * self.V * (2 * self.d + 1)
        fp_roof = {"bound": "alu", "unit": "TFLOP/s", "lanczos_steps_mean": lz_steps / max(nd, 1),
                   "algorithmic_fma_per_site_and_step": 2 * self.d + 1,
                   "achieved": lz_fma * 2.0 / (max(fp_ms, 1e-6) * 1e-3) / 1e12, "peak": peak,
                   "frac": lz_fma * 2.0 / (max(fp_ms, 1e-6) * 1e-3) / 1e12 / peak, "ms": fp_ms}
        return dict(workload=f"{'x'.join(map(str, self.ext))} seed {self.seed}, {self.n} starts", value=su / (step_ms * 1e-3),
                    ms_per_step=step_ms, relax_kernel_ms=relax_ms, first_region_ms=fp_ms,
                    first_region_path="fields of all starts kept, representatives by index" if "g_canon" in out and out["g_canon"] is not None
                    else "representatives re-relaxed",
                    roofline=roof, first_region_roofline=fp_roof, converged_copies_per_s=conv / (step_ms * 1e-3), n_distinct=nd,
                    n_in_first_region=int(st["f"]["n_in_region"].item()),
                    first_region_exceptions=exc_starts[:32], n_exceptions=len(exc_starts),
                    lanczos_unconverged=int((reg & 4).ne(0).sum().item()),
                    mean_sweeps=sweeps_sum / self.n, max_sweeps_seen=int(out["sweeps"].max().item()),
                    gpu_launches=st["launches"]), su, conv, sweeps_sum


def time_pipeline(p, torch, flush, steps, warmup, barrier=None):
    for _ in range(warmup):
        p.step()
        flush.fill_(1)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    relax_ms, fp_ms = [], []
    for k in range(steps):
        ev[k][0].record()
        p.step()
        ev[k][1].record()
        ev[k][1].synchronize()
        relax_ms.append(p.ev[0].elapsed_time(p.ev[1]))
        fp_ms.append(p.fev[0].elapsed_time(p.fev[1]))
        flush.fill_(k & 1)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    per_step = [a.elapsed_time(z) for a, z in ev]
    time_pipeline.last_per_step = per_step      # the `configs` section reports the median step (few repetitions, one hiccup would show)
    return sum(per_step), float(np.mean(relax_ms)), float(np.mean(fp_ms))


def ensemble_config3(b, torch, flush, steps, warmup, peak_dfma, sm_clock_mhz, sms):
    """Config 3 (8 hot 4^3 orbits, 2^20 starts each) as ONE ensemble launch + per-orbit counting and region tests."""
    conf = synth.CONFIGS[3]
    obs = conf["orbits"]
    ext, n = obs[0]["extents"], obs[0]["n_starts"]
    V = synth.volume(ext)
    seeds = [o["seed"] for o in obs]
    ens = b.Ensemble(ext, np.stack([synth.make_theta(o) for o in obs]), seeds)
    kw = dict(omega=conf["omega"], eps=conf["eps"], max_sweeps=conf["max_sweeps"])
    st = {}
    rev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))

    def step():
        rev[0].record()
        r = b.relax_ensemble(ens, n, workspace=st.get("ws"), **kw)
        rev[1].record()
        launches = b.last_launch_count()
        st["ws"] = r["workspace"]
        c = b.count_copies_ensemble(r["F_norm"], r["sig"], r["status"], workspace=st.get("cws"))
        launches += b.last_launch_count()
        st["cws"] = c["workspace"]
        nds = c["n_distinct"].cpu().tolist()
        n_in, exc = [], []
        for k, nd in enumerate(nds):
            member = ens.orbit(k)
            rr = b.relax_batch(member, seeds[k], 0, start_ids=c["rep"][k][:nd].contiguous(), want_g=True, **kw)
            launches += b.last_launch_count()
            f = b.check_fp(member, rr["g_canon"])
            launches += b.last_launch_count()
            st.setdefault("f", {})[k] = (f, c["rep"][k][:nd])
        st.update(r=r, c=c, nds=nds, launches=launches)

    for _ in range(warmup):
        step()
        flush.fill_(1)
    torch.cuda.synchronize()
    ms, rms = [], []
    for k in range(steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step()
        e1.record()
        e1.synchronize()
        ms.append(e0.elapsed_time(e1))
        rms.append(rev[0].elapsed_time(rev[1]))
        flush.fill_(k & 1)
    r = st["r"]
    # the paper's ensemble read-outs (Tab. I / III) of this launch, through the C-ABI; 8 orbits at omega = 1.7 against the
    # paper's 100 orbits at omega = 1: context, not a target
    n_in_dev = torch.tensor([int(st["f"][k][0]["n_in_region"].item()) for k in range(len(seeds))], dtype=torch.int64, device="cuda")
    es = b.ensemble_stats(len(seeds), n, r["F_norm"], st["c"]["rep"], st["c"]["n_distinct"], n_in_dev)["stats"].cpu().tolist()
    sweeps = r["sweeps"].sum(dim=1, dtype=torch.int64).cpu().tolist()
    su = float(V) * float(sum(sweeps))
    step_ms, relax_ms = float(np.median(ms)), float(np.median(rms))
    n_in = [int(st["f"][k][0]["n_in_region"].item()) for k in range(len(seeds))]
    exc = {int(seeds[k]): st["f"][k][1][torch.nonzero(st["f"][k][0]["region"] != 1).flatten()].cpu().tolist() for k in range(len(seeds))}
    fp64 = su * A_D[3] * 2.0 / (relax_ms * 1e-3) / 1e12
    peak = peak_dfma * 2.0 / 1e12
    pipe = sms * FP64_LANES_PER_SM * sm_clock_mhz * 1e6 * 2.0 / 1e12
    out = dict(workload=f"8 orbits 4x4x4 seeds 3..10, {n} starts each, ONE u1gf_relax_ensemble launch", value=su / (step_ms * 1e-3),
               ms_per_step=step_ms, relax_kernel_ms=relax_ms,
               roofline={"bound": "alu", "achieved": fp64, "peak": peak, "unit": "TFLOP/s", "frac": fp64 / peak,
                         "frac_of_fp64_pipe": fp64 / pipe, "kernel": "lanes_4x4x4_blk4x2x2 (ensemble mode)", "kernel_ms": relax_ms,
                         "kernel_share_of_step": relax_ms / step_ms, "traffic": None},
               converged_copies_per_s=float((r["status"] & 1).eq(0).sum().item()) / (step_ms * 1e-3),
               n_distinct_per_orbit=st["nds"], n_in_first_region_per_orbit=n_in,
               ensemble_stats={"n_distinct_mean": es[0], "n_distinct_std": es[1], "best_x_mean": es[2], "best_x_std": es[3],
                               "n_in_first_region_mean": es[4], "n_in_first_region_std": es[5], "orbits": int(es[7]),
                               "call": "u1gf_ensemble_stats",
                               "paper_context": "Tab. I / III, 4^3, 100 orbits x 4 mebisamples, omega = 1: 394.7 +- 228.3 minima, x_g = 0.338 +- 0.014"},
               dedup="u1gf_count_copies_ensemble, all orbits in one pass",
               first_region_exceptions={k: v for k, v in exc.items() if v},
               mean_sweeps_per_orbit=[s / n for s in sweeps], max_sweeps_per_orbit=r["sweeps"].max(dim=1).values.cpu().tolist(),
               gpu_launches=st["launches"])
    ens.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="u1gf", choices=["u1gf", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE config id (1..5); 4 is the metric's workload")
    ap.add_argument("--orbit", type=int, default=0, help="orbit index inside the config")
    ap.add_argument("--starts", type=int, default=0, help="override the number of starts (debugging only)")
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 generic kernel, 2 streamed kernel with plain loads, 3 TMA-staged streamed kernel (u1gf_set_kernel)")
    ap.add_argument("--eps", type=float, default=0.0, help="override eps (measurement only: with --max-sweeps, a fixed number of sweeps per start)")
    ap.add_argument("--max-sweeps", type=int, default=0, help="override max_sweeps (measurement only)")
    ap.add_argument("--merge-tables", action="store_true", help="run the copy-table merge of the multi-GPU path at N = 1 too")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true", help="skip the `configs` section (BASELINE configs 1-3, 5)")
    args = ap.parse_args()

    ri = shard.rank_info_from_env()
    rank, world, local = ri.rank, ri.world, ri.local_rank
    conf, ob = workload(args.config, args.orbit, args.starts)
    if args.eps or args.max_sweeps:
        conf = dict(conf, eps=args.eps or conf["eps"], max_sweeps=args.max_sweeps or conf["max_sweeps"])
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
        # a step of this arm is a bounded sample of the workload: ms_per_step is the time actually spent per step (what the
        # driver's clock sees), ms_per_full_step the time all n starts would take at the measured rate
        full_ms = 1e3 * (sum(dts) / len(dts)) * n / last["sample_starts"]
        print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": 0,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(dts) / len(dts),
                          "ms_per_full_step": full_ms,
                          "ms_per_step_note": "a step is a bounded sample of the workload (cpu_baseline.sample); ms_per_full_step extrapolates it to all starts at the measured rate",
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
    first, _ = shard.weak_start_range(rank, world, n)   # disjoint start ranges of the same orbit, no data-path collective
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    sms = torch.cuda.get_device_properties(local).multi_processor_count

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
            torch.cuda.synchronize()

    pipe = Pipeline(b, torch, conf, ob, first, kernel=args.kernel)
    sampler = ClockSampler(local)
    for _ in range(args.warmup):
        pipe.step()
        flush.fill_(1)
    barrier()
    if rank == 0:
        sampler.start()
    total_ms, relax_ms, fp_ms = time_pipeline(pipe, torch, flush, args.steps, 0, barrier)
    clocks = sampler.stop() if rank == 0 else None
    sm_clock = (clocks or {}).get("sm_mhz") or 1965.0

    # roofline denominators: the in-run DFMA microbenchmark (libu1gf_measure.so) and the driver's HBM figure
    peak_dfma = b.measure_fp64_peak(300.0)
    hbm_peak, hbm_how = 6650.0, "fallback of B200_PROFILING.md"
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            hbm_peak, hbm_how = float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json"
    except (OSError, KeyError, ValueError):
        pass
    main_sum, su_rank, conv, sweeps_sum = pipe.summary(relax_ms, fp_ms, total_ms / args.steps, peak_dfma, sm_clock, sms, hbm_peak)
    total_ms, (sweeps_all, conv_all) = shard.aggregate(total_ms, [sweeps_sum, conv], dist, device="cuda")
    ms_per_step = total_ms / args.steps
    site_updates = float(V) * float(sweeps_all)              # per step, all ranks
    value = site_updates / (ms_per_step * 1e-3)

    # N > 1: the ranks' copy tables merged into the job's table, outside the timed region: all-gather of
    # {F, signature, global first start, multiplicity} of the representatives, then u1gf_merge_copy_tables on every rank
    n_distinct_global = None
    if world > 1 or args.merge_tables:
        st = pipe.state
        nd = st["n_distinct"]
        rep = st["c"]["rep"][:nd]
        F, S, fs, mu, offs = shard.gather_copy_tables(pipe.out["F_norm"][rep], pipe.out["sig"][rep], rep + first,
                                                      st["c"]["multiplicity"][:nd], dist)
        mg = b.merge_copy_tables(F, S, fs, mu)
        n_distinct_global = int(mg["n_merged"].item())

    # e2e: the whole path through u1gf_pipeline_host: link angles in (u1gf_create_orbit), host result arrays out
    e2e = None
    if not args.no_e2e:
        hb = b.host_buffers(n)   # pinned result arrays, made once: the timed region holds copies, not page faults
        th = pipe.theta
        kw = pipe.kw

        def host_step():
            orb = b.Orbit(ext, th)
            orb.set_kernel(args.kernel)
            p = b.pipeline_host(orb, seed, n, first_start=first, nbins=10000, out=hb, **kw)
            nd = p["n_distinct"]
            h2d = th.nbytes
            d2h = n * (8 + 4 + 1 + 32 + 4) + 8 + nd * (8 + 8 + 8 + 8 + 1) + 10000 * 8 + 8 * (1 + (nd + 0) // max(1, (1 << 30) // (V * 16)))
            orb.close()
            return float(V) * float(p["sweeps"].sum(dtype=np.int64)), h2d, d2h
        host_step()
        barrier()
        t0 = time.perf_counter()
        su_e = 0.0
        reps = max(1, args.steps)
        for _ in range(reps):
            su, h2d, d2h = host_step()
            su_e += su
        barrier()
        dt = time.perf_counter() - t0
        te = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if dist:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": su_e * world / float(te[0]), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "repetitions": reps, "call": "u1gf_create_orbit + u1gf_pipeline_host",
               "timing": "wall clock around the synchronous calls, max over ranks"}
        b.lib().u1gf_release_host_scratch()

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0

    rate_rrr = b.measure_fp64_rate(1, 100.0)   # DFMA with three distinct register operands
    rate_mac = b.measure_fp64_rate(2, 100.0)   # the complex multiply-accumulate pattern of w_i
    rate_dmma = b.measure_fp64_rate(6, 100.0)  # the FP64 pipe through DMMA: 64 lanes x SMs x clock
    roofline = main_sum["roofline"]
    roofline.update({"peak_source": "in-run u1gf_measure_fp64_peak (DFMA stream, constant multiplicands), kernel timed alone",
                     "dmma_rate": rate_dmma * 2.0 / 1e12, "frac_of_dmma_rate": roofline.get("achieved", 0.0) / (rate_dmma * 2.0 / 1e12)
                     if roofline["bound"] == "alu" else None,
                     "dfma_rate_3_register_operands": rate_rrr * 2.0 / 1e12, "dfma_rate_complex_mac": rate_mac * 2.0 / 1e12,
                     "hbm_peak_source": hbm_how,
                     "traffic_note": ("traffic is null: the relaxation state never leaves the SM; ncu on 262144 starts of this orbit "
                                      "(profiles/r02_ncu_summaries.md): 13.6 MB DRAM read + 1.96 GB written per launch = 7.5 KB per start "
                                      "(start / dump rings and outputs) against 1.2e4 site updates per start"),
                     "note": ("achieved = site-updates x (8d+16 = %d algorithmic FP64 instructions) x 2 flop / kernel time "
                              "(CUDA events on the launching stream around u1gf_relax_batch); frac = against the DFMA "
                              "microbenchmark, frac_of_fp64_pipe / frac_of_dmma_rate = against 64 lanes x SMs x clock, which "
                              "only DMMA reaches (DESIGN.md section 7.1)") % A_D[d]})

    configs = None
    if not args.no_all_configs and world == 1 and not args.starts and not args.eps and not args.max_sweeps:
        configs = {}
        csteps, cwarm = 3, 1
        for cid, oi in [(1, 0), (2, 0)] + [(5, k) for k in range(5)]:
            c2, o2 = workload(cid, oi, 0)
            p2 = Pipeline(b, torch, c2, o2, 0)
            t_ms, r_ms, f_ms = time_pipeline(p2, torch, flush, csteps, cwarm + (1 if cid == 5 and oi >= 2 else 0))
            s2, _, _, _ = p2.summary(r_ms, f_ms, float(np.median(time_pipeline.last_per_step)), peak_dfma, sm_clock, sms, hbm_peak)
            s2.update(steps=csteps, warmup=cwarm, ms_per_step_is="median of the timed steps")
            if cid == 5 and oi == 2:
                # the one-call host API on a hot orbit (most starts are their own copy): the handle's second and later calls
                # keep the fields of all starts from the first pass instead of relaxing the representatives again
                n2, V2 = o2["n_starts"], synth.volume(o2["extents"])
                hb2 = b.host_buffers(n2)
                orb2 = b.Orbit(o2["extents"], p2.theta)
                kw2 = dict(p2.kw, nbins=10000, out=hb2)
                b.pipeline_host(orb2, o2["seed"], n2, **kw2)      # first call on the handle: learns that the orbit is hot
                b.pipeline_host(orb2, o2["seed"], n2, **kw2)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                for _ in range(csteps):
                    ph = b.pipeline_host(orb2, o2["seed"], n2, **kw2)
                dt = (time.perf_counter() - t0) / csteps
                su2 = float(V2) * float(ph["sweeps"].sum(dtype=np.int64))
                nd2 = ph["n_distinct"]
                s2["e2e"] = {"value": su2 / dt, "unit": UNIT, "ms_per_call": dt * 1e3, "fraction_of_value": su2 / dt / s2["value"],
                             "h2d_bytes_per_step": 0, "d2h_bytes_per_step": int(n2 * (8 + 4 + 1 + 32 + 4) + 16 + nd2 * 33 + 80000),
                             "call": "u1gf_pipeline_host on an existing handle (third and later calls), pinned per-start arrays",
                             "gpu_launches": b.last_launch_count(), "n_distinct": nd2, "n_in_first_region": ph["n_in_region"]}
                del hb2, orb2, ph
                b.lib().u1gf_release_host_scratch()
            configs[f"cfg{cid}_{'x'.join(map(str, o2['extents']))}"] = s2
            del p2
            torch.cuda.empty_cache()
        # the paper's other volumes (Tab. I, Tab. III): hot orbits, seed 21, not BASELINE configs
        for ext2, n2 in (((10, 10), 1 << 20), ((6, 6, 6), 1 << 20), ((8, 8, 8), 1 << 18)):
            c2 = dict(name="paper_volume", omega=1.7, eps=1e-13, max_sweeps=20000)
            o2 = dict(extents=ext2, kind="uniform", seed=21, n_starts=n2)
            p2 = Pipeline(b, torch, c2, o2, 0)
            t_ms, r_ms, f_ms = time_pipeline(p2, torch, flush, csteps, cwarm + 1)
            s2, _, _, _ = p2.summary(r_ms, f_ms, float(np.median(time_pipeline.last_per_step)), peak_dfma, sm_clock, sms, hbm_peak)
            s2.update(steps=csteps, warmup=cwarm + 1, ms_per_step_is="median of the timed steps")
            configs[f"paper_volume_{'x'.join(map(str, ext2))}"] = s2
            del p2
            torch.cuda.empty_cache()
        configs["cfg3_ensemble"] = ensemble_config3(b, torch, flush, csteps, cwarm, peak_dfma, sm_clock, sms)

    cpu = None
    if not args.no_cpu_baseline:
        cpu, _, _ = oracle_leg(conf, ob, 10.0)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config, "clocks": clocks, "e2e": e2e, "gpu_launches": main_sum["gpu_launches"],
            "gpu_launches_note": "kernels of libu1gf.so per step, counted by the library; CUB's sort/scan launches inside u1gf_count_copies are extra",
            "roofline": roofline, "cpu_baseline": cpu,
            "converged_copies_per_s": conv_all / (ms_per_step * 1e-3), "n_distinct": main_sum["n_distinct"],
            "n_distinct_all_ranks_merged": n_distinct_global,
            "n_in_first_region": main_sum["n_in_first_region"], "first_region_exceptions": main_sum["first_region_exceptions"],
            "first_region_roofline": main_sum["first_region_roofline"],
            "mean_sweeps": sweeps_all / (n * world), "max_sweeps_seen": main_sum["max_sweeps_seen"], "configs": configs}
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
